// adsc_exp.cuh — branch-free fp64 exponential used by the stage kernels (resident and persistent
// streaming): e^{-delta} of eqs (2), (3) is the only transcendental on the hot path.
#pragma once

namespace adsc {

// exp coefficients (read as constant-bank operands)
static __constant__ double c_exp[18] = {
    1.4426950408889634074,            // 0  log2 e
    6755399441055744.0,               // 1  1.5 * 2^52 (round-to-nearest-integer shift)
    -6.93147180369123816490e-01,      // 2  -ln2 (high part)
    -1.90821492927058770002e-10,      // 3  -ln2 (low part)
    1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0, 1.0 / 5040.0, 1.0 / 40320.0,   // 4..10: 1/k!, k=2..8
    1.0 / 362880.0, 1.0 / 3628800.0, 1.0 / 39916800.0, 1.0 / 479001600.0, 1.0 / 6227020800.0,  // 11..15: k=9..13
    -708.0, 709.0                     // 16, 17 clamps
};

// Branch-free e^x (x clamped to [-708, 709]; NaN propagates; e^0 = 1 exactly): k = rint(x log2 e),
// r = x - k ln 2 in two pieces, Taylor polynomial of degree 13 split in two halves to shorten the
// dependency chain (|r| <= 0.347: truncation r^14/14! < 5e-18), scaled by 2^k through the exponent field.
__device__ __forceinline__ double exp3_ref(double x)
{
    x = (x < c_exp[16]) ? c_exp[16] : x;
    x = (x > c_exp[17]) ? c_exp[17] : x;
    const double t = fma(x, c_exp[0], c_exp[1]);
    const int k = __double2loint(t);
    const double kf = t - c_exp[1];
    double r = fma(kf, c_exp[2], x);
    r = fma(kf, c_exp[3], r);
    double lo = fma(r, c_exp[8], c_exp[7]);
    double hi = fma(r, c_exp[15], c_exp[14]);
    const double r2 = r * r;
    lo = fma(r, lo, c_exp[6]);        hi = fma(r, hi, c_exp[13]);
    const double r3 = r2 * r, r4 = r2 * r2;
    lo = fma(r, lo, c_exp[5]);        hi = fma(r, hi, c_exp[12]);
    const double r7 = r4 * r3;
    lo = fma(r, lo, c_exp[4]);        hi = fma(r, hi, c_exp[11]);
    lo = fma(r, lo, 1.0);             hi = fma(r, hi, c_exp[10]);
    lo = fma(r, lo, 1.0);             hi = fma(r, hi, c_exp[9]);
    const double e = fma(r7, hi, lo);
    return e * __hiloint2double((k + 1023) << 20, 0);
}

// e^{x_p} for P values that lie close together: one exp at the reference x_{P-1}, the rest
// relative to it.  exp(z) = 1 + z t(z), t = sum_{k<=5} z^k/(k+1)!; for |z| <= 2^-6 the truncation
// is z^7/5040 < 5e-17 relative.  x = 0 gives exactly 1 (pure AdS stays bit-exact).
// `scale` multiplies every result (one extra multiplication: it is folded into the reference value).
// SHIFTED: every argument is x_p + shift; the differences do not contain the shift, so it is added to the
// reference argument only (and to every argument if full evaluations are needed) -- the caller may have `shift`
// ready much later than x.
// tier (self-test only): 0, 1, 2 = 2, 3, 5 terms of t; 3 = a full evaluation per point.
// WARP: the number of terms is chosen for the whole warp (the largest spread of its 32 threads), so that the warp does
// not execute two branches one after the other when its lanes disagree; every lane of the warp must make the call.
template <int P, bool SCALED = false, bool SHIFTED = false, bool WARP = false>
__device__ __forceinline__ void exp3_near(const double (&x)[P], double (&E)[P], const double scale = 1.0, int *tier = nullptr,
                                          const double shift = 0.0)
{
    const double xr = x[P - 1];
    double z[P];
    int hmax = 0;                            // largest |z| of the thread (of the warp), as the high word of the double
#pragma unroll
    for (int p = 0; p < P - 1; ++p) {
        z[p] = x[p] - xr;
        hmax = max(hmax, __double2hiint(z[p]) & 0x7fffffff);
    }
    if (WARP) hmax = __reduce_max_sync(0xffffffffu, hmax);
    const int big = hmax > 0x3f900000;       // |z| > 2^-6 (or NaN)
    const int mid = hmax > 0x3f500000;       // |z| > 2^-10
    const int sml = hmax > 0x3f100000;       // |z| > 2^-14
    const double xs = SHIFTED ? xr + shift : xr;
    const double Er = SCALED ? exp3_ref(xs) * scale : exp3_ref(xs);
    E[P - 1] = Er;
    if (tier) *tier = sml + mid + big;       // which branch below runs (adsc_selftest_exp only; folds away otherwise)
    if (!sml) {                              // |z| <= 2^-14: two terms of t suffice (z^4/24 < 6e-19)
#pragma unroll
        for (int p = 0; p < P - 1; ++p) {
            double t = fma(z[p], c_exp[5], c_exp[4]);
            t = fma(z[p], t, 1.0);
            E[p] = fma(Er * z[p], t, Er);
        }
    } else if (!mid) {                       // |z| <= 2^-10: three terms of t suffice (z^5/120 < 8e-18)
#pragma unroll
        for (int p = 0; p < P - 1; ++p) {
            double t = fma(z[p], c_exp[6], c_exp[5]);
            t = fma(z[p], t, c_exp[4]);
            t = fma(z[p], t, 1.0);
            E[p] = fma(Er * z[p], t, Er);
        }
    } else if (!big) {
#pragma unroll
        for (int p = 0; p < P - 1; ++p) {
            double t = fma(z[p], c_exp[8], c_exp[7]);
            t = fma(z[p], t, c_exp[6]);
            t = fma(z[p], t, c_exp[5]);
            t = fma(z[p], t, c_exp[4]);
            t = fma(z[p], t, 1.0);
            E[p] = fma(Er * z[p], t, Er);
        }
    } else {
#pragma unroll
        for (int p = 0; p < P - 1; ++p) {
            const double xp = SHIFTED ? x[p] + shift : x[p];
            E[p] = SCALED ? exp3_ref(xp) * scale : exp3_ref(xp);
        }
    }
}

}  // namespace adsc
