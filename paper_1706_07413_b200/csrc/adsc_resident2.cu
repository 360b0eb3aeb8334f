// adsc_resident2.cu — resident RK4 kernel, second generation ("v2"): one ensemble member per
// CTA (or per cluster of CL CTAs), the whole state on chip across all RK stages and steps.
//
// What changed against adsc_resident.cu (v1), and why (profiles/r01_v1_resident.md):
//   * TWO barriers per RK stage instead of three.  The delta quadrature (SURVEY.md 8(a) a1-a2,
//     eq (6)) is used in its telescoped form
//         delta_i = h * S_{i+2} + (h/24) (25 f_{i+1} + 12 f_i - f_{i-1}),   S_j = sum_{m>=j} f_m (+ top term)
//     which is the same sum of 4-point increments I_k re-associated.
//     A thread's scan element is then the plain sum of its OWN f values, so the scan partials are
//     published together with the new stage state, through the same barrier.
//   * Cluster barriers are split (arrive.release / wait.acquire) and independent arithmetic
//     (Kreiss-Oliger terms, interior stencils, RK accumulators) sits between arrive and wait.
//   * One full exp per thread; the other P-1 points use exp(z) for |z| <= 2^-6 by a degree-6
//     polynomial relative to that reference (full exp again whenever the bound fails).
//   * The second scan level is a uniform loop over the published warp totals (no second shuffle scan).
//
// Per RK stage (equations PAPER.md:43-53 eqs (2)-(6); boundary conditions PAPER.md:59-75):
//   phase 1  (needs neighbours' Phi, Pi edges + scan partials)  delta, E = e^{-delta}, fluxes G, H, F,
//            eq (4) for A with its RK combine, publish H, F edges                      -> barrier F
//   phase 2  Kreiss-Oliger Q Phi, Q Pi and interior D4 (before the wait), edge D4, RK combine for
//            Phi, Pi, collapse test (stage 4), f of the NEW state, thread/warp scan,
//            publish Phi, Pi edges + warp totals                                       -> barrier S
#include <cooperative_groups.h>

#include "adsc_internal.cuh"
#include "adsc_resident.cuh"

namespace cg = cooperative_groups;

namespace adsc {

template <int P, int THREADS, bool ACC_REG>
struct Res2Layout {
    static constexpr int SEG = P * THREADS;
    static constexpr int LD = THREADS + 2;          // halo column on each side
    static constexpr int NW = THREADS / 32;
    static constexpr int RX = (P < 6) ? P : 6;      // rows of the state exchange buffers
    static constexpr int o_xPhi = 0;
    static constexpr int o_xPi = o_xPhi + RX * LD;
    static constexpr int o_xH = o_xPi + RX * LD;
    static constexpr int o_xF = o_xH + 4 * LD;
    static constexpr int o_tSC = o_xF + 4 * LD;      // -2 sin x cos x, [P][LD] with halo columns
    static constexpr int o_tT = o_tSC + P * LD;      // tan^2 x
    static constexpr int o_tC = o_tT + P * THREADS;  // cot^2 x / (12 h)
    static constexpr int o_un = o_tC + P * THREADS;
    static constexpr int o_acc = o_un + 3 * P * THREADS;
    static constexpr int o_wtot = o_acc + (ACC_REG ? 0 : 3 * P * THREADS);
    static constexpr int o_flag = o_wtot + 64;
    static constexpr int n_doubles = o_flag + 2;
    static constexpr size_t bytes = (size_t)n_doubles * sizeof(double);
};

// Branch-free e^x (x clamped to [-708, 709]; NaN propagates; e^0 = 1 exactly): k = rint(x log2 e),
// r = x - k ln 2 in two pieces, Taylor polynomial of degree 13 split in two halves to shorten the
// dependency chain (|r| <= 0.347: truncation r^14/14! < 5e-18), scaled by 2^k through the exponent field.
__device__ __forceinline__ double exp_ref(double x)
{
    x = (x < -708.0) ? -708.0 : x;
    x = (x > 709.0) ? 709.0 : x;
    const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
    const int k = __double2loint(t);
    const double kf = t - 6755399441055744.0;
    double r = fma(kf, -6.93147180369123816490e-01, x);
    r = fma(kf, -1.90821492927058770002e-10, r);
    double lo = fma(r, 1.0 / 720.0, 1.0 / 120.0);
    double hi = fma(r, 1.0 / 6227020800.0, 1.0 / 479001600.0);
    const double r2 = r * r;
    lo = fma(r, lo, 1.0 / 24.0);      hi = fma(r, hi, 1.0 / 39916800.0);
    const double r3 = r2 * r, r4 = r2 * r2;
    lo = fma(r, lo, 1.0 / 6.0);       hi = fma(r, hi, 1.0 / 3628800.0);
    const double r7 = r4 * r3;
    lo = fma(r, lo, 0.5);             hi = fma(r, hi, 1.0 / 362880.0);
    lo = fma(r, lo, 1.0);             hi = fma(r, hi, 1.0 / 40320.0);
    lo = fma(r, lo, 1.0);             hi = fma(r, hi, 1.0 / 5040.0);
    const double e = fma(r7, hi, lo);
    return e * __hiloint2double((k + 1023) << 20, 0);
}

// e^{x_p} for P values that lie close together: one exp at the reference x_{P-1}, the rest
// relative to it.  exp(z) = 1 + z t(z), t = sum_{k<=5} z^k/(k+1)!; for |z| <= 2^-6 the truncation
// is z^7/5040 < 5e-17 relative.  x = 0 gives exactly 1 (pure AdS stays bit-exact).
template <int P>
__device__ __forceinline__ void exp_near(const double (&x)[P], double (&E)[P])
{
    const double xr = x[P - 1];
    double z[P];
    int big = 0;
#pragma unroll
    for (int p = 0; p < P - 1; ++p) {
        z[p] = x[p] - xr;
        big |= ((__double2hiint(z[p]) & 0x7fffffff) > 0x3f900000) ? 1 : 0;    // |z| > 2^-6 (or NaN)
    }
    const double Er = exp_ref(xr);
    E[P - 1] = Er;
    if (!big) {
#pragma unroll
        for (int p = 0; p < P - 1; ++p) {
            double t = fma(z[p], 1.0 / 720.0, 1.0 / 120.0);
            t = fma(z[p], t, 1.0 / 24.0);
            t = fma(z[p], t, 1.0 / 6.0);
            t = fma(z[p], t, 0.5);
            t = fma(z[p], t, 1.0);
            E[p] = fma(Er * z[p], t, Er);
        }
    } else {
#pragma unroll
        for (int p = 0; p < P - 1; ++p) E[p] = exp_ref(x[p]);
    }
}

__device__ __forceinline__ void cluster_arrive()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_wait()
{
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int P, int THREADS, bool ACC_REG, bool MULTI>
__global__ void __launch_bounds__(THREADS, 1) k_resident2(const ResParams prm)
{
    using L = Res2Layout<P, THREADS, ACC_REG>;
    constexpr int LD = L::LD, NW = L::NW, SEG = L::SEG, RX = L::RX;
    extern __shared__ __align__(16) double smem[];
    double *xPhi = smem + L::o_xPhi, *xPi = smem + L::o_xPi, *xH = smem + L::o_xH, *xF = smem + L::o_xF;
    double *tSC = smem + L::o_tSC, *tT = smem + L::o_tT, *tC = smem + L::o_tC;
    double *un = smem + L::o_un, *accS = smem + L::o_acc, *wtot = smem + L::o_wtot;
    int *iflag = reinterpret_cast<int *>(smem + L::o_flag);

    cg::cluster_group cluster = cg::this_cluster();
    const int CL = MULTI ? prm.CL : 1;
    const int rank = MULTI ? (int)cluster.block_rank() : 0;
    const int b = blockIdx.x / CL;
    MemberRec *rec = prm.rec + b;
    if (rec->collapsed || prm.nsteps <= 0) return;      // uniform over the cluster

    const Problem &pb = prm.pb;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, col = tid + 1;
    const int g0 = rank * SEG + tid * P;                 // first owned grid index
    const bool lo_edge = (tid == 0), hi_edge = (tid == THREADS - 1);
    const bool first = lo_edge && rank == 0;             // owns i = 0
    const bool last = hi_edge && rank == CL - 1;         // owns i = N-2; i = N-1 is its halo
    const int gw = rank * NW + warp, NG = NW * CL;       // my warp / number of warps per member
    const size_t row = (size_t)b * pb.NP;

    double *nb_lo_xPhi = nullptr, *nb_lo_xPi = nullptr, *nb_lo_xH = nullptr, *nb_lo_xF = nullptr;
    double *nb_hi_xPhi = nullptr, *nb_hi_xPi = nullptr, *nb_hi_xH = nullptr, *nb_hi_xF = nullptr;
    if (MULTI) {
        if (rank > 0) {
            nb_lo_xPhi = cluster.map_shared_rank(xPhi, rank - 1); nb_lo_xPi = cluster.map_shared_rank(xPi, rank - 1);
            nb_lo_xH = cluster.map_shared_rank(xH, rank - 1); nb_lo_xF = cluster.map_shared_rank(xF, rank - 1);
        }
        if (rank < CL - 1) {
            nb_hi_xPhi = cluster.map_shared_rank(xPhi, rank + 1); nb_hi_xPi = cluster.map_shared_rank(xPi, rank + 1);
            nb_hi_xH = cluster.map_shared_rank(xH, rank + 1); nb_hi_xF = cluster.map_shared_rank(xF, rank + 1);
        }
    }

    const double d4c = 1.0 / (12.0 * pb.h), koc = pb.ko_eps / (64.0 * pb.h);
    const double hh = 0.5 * pb.h, c25 = 25.0 * pb.h / 48.0, c12 = 0.25 * pb.h, c1 = pb.h / 48.0;
    const double thr = pb.thr;
    const double dt_half = 0.5 * pb.dt, dt_6 = pb.dt / 6.0, dt_3 = pb.dt / 3.0;
    const double inv12h2 = 1.0 / (12.0 * pb.h * pb.h), c_org = 1.0 / (2.0 * pb.h);

    // ---- load: own points to registers, u^n and tables to shared memory
    double ph[P], pi[P], a[P];
    double accP[ACC_REG ? P : 1], accQ[ACC_REG ? P : 1], accA[ACC_REG ? P : 1];
    {
        const double2 *s0 = reinterpret_cast<const double2 *>(prm.U[0] + row + g0);
        const double2 *s1 = reinterpret_cast<const double2 *>(prm.U[1] + row + g0);
        const double2 *s2 = reinterpret_cast<const double2 *>(prm.U[2] + row + g0);
#pragma unroll
        for (int p = 0; p < P; p += 2) {
            double2 v0 = s0[p / 2], v1 = s1[p / 2], v2 = s2[p / 2];
            ph[p] = v0.x; ph[p + 1] = v0.y; pi[p] = v1.x; pi[p + 1] = v1.y; a[p] = v2.x; a[p + 1] = v2.y;
        }
#pragma unroll
        for (int p = 0; p < P; ++p) {
            un[(0 * P + p) * THREADS + tid] = ph[p];
            un[(1 * P + p) * THREADS + tid] = pi[p];
            un[(2 * P + p) * THREADS + tid] = a[p];
            tSC[p * LD + col] = -2.0 * prm.tb.sc[g0 + p];
            tT[p * THREADS + tid] = prm.tb.T[g0 + p];
            tC[p * THREADS + tid] = prm.tb.C[g0 + p] * d4c;
            if constexpr (ACC_REG) { accP[p] = ph[p]; accQ[p] = pi[p]; accA[p] = a[p]; }
            else { accS[(0 * P + p) * THREADS + tid] = ph[p]; accS[(1 * P + p) * THREADS + tid] = pi[p]; accS[(2 * P + p) * THREADS + tid] = a[p]; }
        }
        if (lo_edge) tSC[(P - 1) * LD + 0] = -2.0 * prm.tb.sc[g0 - 1];            // odd ghost at x=0
        if (hi_edge) tSC[0 * LD + THREADS + 1] = -2.0 * prm.tb.sc[g0 + P];        // 0 at x=pi/2
        if (tid < 2) iflag[tid] = 0;
    }

    // Kept across barrier S: f' = -2 f of the own points (fo), thread-local suffix sums s_p
    // (so; s_P = top term), the exclusive warp-level suffix (excl), and the own-point part of the
    // Kreiss-Oliger sums of the state just completed (kP, kQ).
    double fo[P], so[P], excl, kP[P], kQ[P];
    const double kw0 = -20.0 * koc, kw1 = 15.0 * koc, kw2 = -6.0 * koc, kw3 = koc;
    auto kow = [&](int j) { return j == 0 ? kw0 : (j == 1 ? kw1 : (j == 2 ? kw2 : kw3)); };

    // f', s of the new state; publish the state edges (stores go out before the shuffle chain).
    auto state_sums_and_edges = [&]() {
#pragma unroll
        for (int p = 0; p < P; ++p) fo[p] = tSC[p * LD + col] * fma(ph[p], ph[p], pi[p] * pi[p]);
        // top term of the telescoped rule: S_{N-1} = S_N = f_{N-2}/12 (f_N = -f_{N-2}, f_{N-1} = 0)
        so[P - 1] = fo[P - 1] + (last ? fo[P - 1] * (1.0 / 12.0) : 0.0);
#pragma unroll
        for (int p = P - 2; p >= 0; --p) so[p] = so[p + 1] + fo[p];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            xPhi[k * LD + col] = ph[k]; xPi[k * LD + col] = pi[k];
            xPhi[(RX - 3 + k) * LD + col] = ph[P - 3 + k]; xPi[(RX - 3 + k) * LD + col] = pi[P - 3 + k];
        }
        if (lo_edge) {
            if (rank == 0) {            // x=0: Phi odd, Pi even (R2)
#pragma unroll
                for (int k = 1; k <= 3; ++k) { xPhi[(RX - k) * LD] = -ph[k]; xPi[(RX - k) * LD] = pi[k]; }
            } else if (MULTI) {
#pragma unroll
                for (int k = 0; k < 3; ++k) { nb_lo_xPhi[k * LD + THREADS + 1] = ph[k]; nb_lo_xPi[k * LD + THREADS + 1] = pi[k]; }
            }
        }
        if (hi_edge) {
            if (rank == CL - 1) {       // x=pi/2: Phi even, Pi odd, Dirichlet values (R3, eqs 9, 10)
                xPhi[0 * LD + THREADS + 1] = 0.0;        xPi[0 * LD + THREADS + 1] = 0.0;
                xPhi[1 * LD + THREADS + 1] = ph[P - 1];  xPi[1 * LD + THREADS + 1] = -pi[P - 1];
                xPhi[2 * LD + THREADS + 1] = ph[P - 2];  xPi[2 * LD + THREADS + 1] = -pi[P - 2];
            } else if (MULTI) {
#pragma unroll
                for (int k = 0; k < 3; ++k) { nb_hi_xPhi[(RX - 3 + k) * LD] = ph[P - 3 + k]; nb_hi_xPi[(RX - 3 + k) * LD] = pi[P - 3 + k]; }
            }
        }
    };
    // a2, warp level: inclusive suffix over the lanes, publish the warp total.
    auto warp_scan_publish = [&]() {
        const double incl = warp_suffix_incl(so[0]);
        excl = incl - so[0];
        const double wsum = __shfl_sync(0xffffffffu, incl, 0);
        if (MULTI) {
            if (lane < CL) cluster.map_shared_rank(wtot, lane)[gw] = wsum;
        } else {
            if (lane == 0) wtot[gw] = wsum;
        }
    };
    // Own-point part of Q Phi, Q Pi (R6) of the state in ph, pi; the halo part is added after barrier S.
    auto ko_own = [&]() {
#pragma unroll
        for (int p = 0; p < P; ++p) {
            double sP = kw0 * ph[p], sQ = kw0 * pi[p];
#pragma unroll
            for (int j = 1; j <= 3; ++j) {
                if (p - j >= 0) { sP = fma(kow(j), ph[p - j], sP); sQ = fma(kow(j), pi[p - j], sQ); }
                if (p + j < P)  { sP = fma(kow(j), ph[p + j], sP); sQ = fma(kow(j), pi[p + j], sQ); }
            }
            kP[p] = sP; kQ[p] = sQ;
        }
    };
    auto arrive = [&]() { if (MULTI) cluster_arrive(); };
    auto wait = [&]() { if (MULTI) cluster_wait(); else __syncthreads(); };

    state_sums_and_edges();
    warp_scan_publish();
    arrive();
    ko_own();
    wait();

    long long n_done = 0;
    int collapsed = 0;
#pragma unroll 1
    for (long long n = 0; n < prm.nsteps; ++n) {
#pragma unroll 1
        for (int s = 0; s < 4; ++s) {
            const double a_next = (s == 2) ? pb.dt : dt_half;
            const double b_w = (s == 0 || s == 3) ? dt_6 : dt_3;

            // ---------------------------------------------------------------- phase 1 (after barrier S)
            double hlP[3], hrP[3], hlQ[3], hrQ[3];    // 3 halo points per side of the stage state
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                hlP[k] = xPhi[(RX - 3 + k) * LD + col - 1]; hlQ[k] = xPi[(RX - 3 + k) * LD + col - 1];
                hrP[k] = xPhi[k * LD + col + 1];            hrQ[k] = xPi[k * LD + col + 1];
            }
            const double scm = tSC[(P - 1) * LD + col - 1], scp = tSC[0 * LD + col + 1];
            // a2, member level: all f' above this thread's points
            double B0 = excl, B1 = 0.0;
            {
                int w = gw + 1;
                for (; w + 1 < NG; w += 2) { B0 += wtot[w]; B1 += wtot[w + 1]; }
                if (w < NG) B0 += wtot[w];
            }
            const double B = B0 + B1;
            // halo part of the Kreiss-Oliger sums
#pragma unroll
            for (int p = 0; p < P; ++p) {
#pragma unroll
                for (int j = 1; j <= 3; ++j) {
                    if (p - j < 0) { kP[p] = fma(kow(j), hlP[3 + p - j], kP[p]); kQ[p] = fma(kow(j), hlQ[3 + p - j], kQ[p]); }
                    if (p + j >= P) { kP[p] = fma(kow(j), hrP[p + j - P], kP[p]); kQ[p] = fma(kow(j), hrQ[p + j - P], kQ[p]); }
                }
            }
            // a1/a2: -delta_p = (h/2)(s_{p+2} + B) + (h/48)(25 f'_{p+1} + 12 f'_p - f'_{p-1}),  f' = -2 f
            double nd[P];
            {
                const double fm = scm * fma(hlP[2], hlP[2], hlQ[2] * hlQ[2]);     // f'_{-1}
                const double fp = scp * fma(hrP[0], hrP[0], hrQ[0] * hrQ[0]);     // f'_{P}
                const double top = last ? fo[P - 1] * (1.0 / 12.0) : 0.0;         // as in state_sums_and_edges
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const double f_lo = (p == 0) ? fm : fo[p - 1];
                    const double f_hi = (p == P - 1) ? fp : fo[p + 1];
                    const double s2 = (p + 2 < P) ? so[p + 2] : ((p + 2 == P) ? top : top - fp);
                    double loc = c25 * f_hi;
                    loc = fma(c12, fo[p], loc);
                    loc = fma(-c1, f_lo, loc);
                    nd[p] = fma(hh, s2 + B, loc);
                }
            }
            double E[P];
            exp_near<P>(nd, E);
            // a3 fluxes
            double H[P], F[P], kAv[P], G1 = 0.0, G2 = 0.0, Gl1 = 0.0, Gl2 = 0.0;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const double AE = a[p] * E[p];
                const double G = AE * ph[p];
                H[p] = AE * pi[p];
                F[p] = tT[p * THREADS + tid] * G;
                if (p == 1) G1 = G;
                if (p == 2) G2 = G;
                if (p == P - 1) Gl1 = G;
                if (p == P - 2) Gl2 = G;
                kAv[p] = (tSC[p * LD + col] * a[p]) * (G * pi[p]);        // eq (4): -2 sc A G Pi
            }
            if (first) kAv[0] = 0.0;                                      // A(0,t)=1, eq (8)
            // publish flux edges
            xH[0 * LD + col] = H[0]; xH[1 * LD + col] = H[1]; xH[2 * LD + col] = H[P - 2]; xH[3 * LD + col] = H[P - 1];
            xF[0 * LD + col] = F[0]; xF[1 * LD + col] = F[1]; xF[2 * LD + col] = F[P - 2]; xF[3 * LD + col] = F[P - 1];
            if (lo_edge) {
                if (rank == 0) {       // x=0: H even, F odd
                    xH[2 * LD] = H[2]; xH[3 * LD] = H[1]; xF[2 * LD] = -F[2]; xF[3 * LD] = -F[1];
                } else if (MULTI) {
                    nb_lo_xH[0 * LD + THREADS + 1] = H[0]; nb_lo_xH[1 * LD + THREADS + 1] = H[1];
                    nb_lo_xF[0 * LD + THREADS + 1] = F[0]; nb_lo_xF[1 * LD + THREADS + 1] = F[1];
                }
            }
            if (hi_edge) {
                if (rank == CL - 1) {  // x=pi/2: H odd with H=0 there; F even with the limit of R5
                    xH[0 * LD + THREADS + 1] = 0.0; xH[1 * LD + THREADS + 1] = -H[P - 1];
                    xF[0 * LD + THREADS + 1] = (16.0 * Gl1 - Gl2) * inv12h2;
                    xF[1 * LD + THREADS + 1] = F[P - 1];
                } else if (MULTI) {
                    nb_hi_xH[2 * LD] = H[P - 2]; nb_hi_xH[3 * LD] = H[P - 1];
                    nb_hi_xF[2 * LD] = F[P - 2]; nb_hi_xF[3 * LD] = F[P - 1];
                }
            }
            arrive();                                                     // barrier F

            // ---------------------------------------------------------------- between arrive and wait
            // a4/a5 for A (eq 4 needs no neighbour).  Invariant at the start of every step: acc == u^n == state.
            int bad = 0;
            if (s < 3) {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int ui = (2 * P + p) * THREADS + tid;
                    if constexpr (ACC_REG) accA[p] = fma(b_w, kAv[p], accA[p]);
                    else accS[ui] = fma(b_w, kAv[p], accS[ui]);
                    a[p] = fma(a_next, kAv[p], un[ui]);
                }
            } else {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int ui = (2 * P + p) * THREADS + tid;
                    double accn;
                    if constexpr (ACC_REG) { accn = fma(b_w, kAv[p], accA[p]); accA[p] = accn; }
                    else { accn = fma(b_w, kAv[p], accS[ui]); accS[ui] = accn; }
                    a[p] = accn; un[ui] = accn;
                    if (!(accn >= thr)) bad = 1;
                }
            }
            // interior centred differences (own fluxes only)
            double dH[P], dF[P];
#pragma unroll
            for (int p = 2; p < P - 2; ++p) {
                dH[p] = fma(8.0, H[p + 1] - H[p - 1], H[p - 2] - H[p + 2]);
                dF[p] = fma(8.0, F[p + 1] - F[p - 1], F[p - 2] - F[p + 2]);
            }
            wait();                                                       // barrier F

            // ---------------------------------------------------------------- phase 2
            {
                const double Hm2 = xH[2 * LD + col - 1], Hm1 = xH[3 * LD + col - 1];
                const double Fm2 = xF[2 * LD + col - 1], Fm1 = xF[3 * LD + col - 1];
                const double Hp0 = xH[0 * LD + col + 1], Hp1 = xH[1 * LD + col + 1];
                const double Fp0 = xF[0 * LD + col + 1], Fp1 = xF[1 * LD + col + 1];
                dH[0] = fma(8.0, H[1] - Hm1, Hm2 - H[2]);
                dF[0] = fma(8.0, F[1] - Fm1, Fm2 - F[2]);
                dH[1] = fma(8.0, H[2] - H[0], Hm1 - H[3]);
                dF[1] = fma(8.0, F[2] - F[0], Fm1 - F[3]);
                dH[P - 2] = fma(8.0, H[P - 1] - H[P - 3], H[P - 4] - Hp0);
                dF[P - 2] = fma(8.0, F[P - 1] - F[P - 3], F[P - 4] - Fp0);
                dH[P - 1] = fma(8.0, Hp0 - H[P - 2], H[P - 3] - Hp1);
                dF[P - 1] = fma(8.0, Fp0 - F[P - 2], F[P - 3] - Fp1);
            }
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const double qq = kQ[p];
                kP[p] = fma(d4c, dH[p], kP[p]);
                kQ[p] = fma(tC[p * THREADS + tid], dF[p], qq);
                if (p == 0 && first) {           // Phi(0,t)=0 (eq 7); Pi_dot(0) = 3 (A e^{-delta} Phi)'(0) (R4)
                    kP[0] = 0.0;
                    kQ[0] = fma(8.0 * G1 - G2, c_org, qq);
                }
            }
            // a5: new stage state first (the scan needs it), accumulators after the shuffle chain started
            double kPs[P], kQs[P];
            if (s < 3) {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                    kPs[p] = kP[p]; kQs[p] = kQ[p];
                    ph[p] = fma(a_next, kP[p], un[uP]); pi[p] = fma(a_next, kQ[p], un[uQ]);
                }
            } else {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                    double nP, nQ;
                    if constexpr (ACC_REG) { nP = fma(b_w, kP[p], accP[p]); nQ = fma(b_w, kQ[p], accQ[p]); accP[p] = nP; accQ[p] = nQ; }
                    else { nP = fma(b_w, kP[p], accS[uP]); nQ = fma(b_w, kQ[p], accS[uQ]); accS[uP] = nP; accS[uQ] = nQ; }
                    ph[p] = nP; pi[p] = nQ; un[uP] = nP; un[uQ] = nQ;
                }
            }
            state_sums_and_edges();
            warp_scan_publish();
            const int par = (int)(n & 1);
            if (MULTI && s == 3 && bad) {
                for (int r = 0; r < CL; ++r) cluster.map_shared_rank(iflag, r)[par] = 1;
            }
            arrive();                                                     // barrier S
            if (s < 3) {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                    if constexpr (ACC_REG) { accP[p] = fma(b_w, kPs[p], accP[p]); accQ[p] = fma(b_w, kQs[p], accQ[p]); }
                    else { accS[uP] = fma(b_w, kPs[p], accS[uP]); accS[uQ] = fma(b_w, kQs[p], accS[uQ]); }
                }
            }
            ko_own();                                                     // for the next stage
            if (s == 3) {
                // a6: collapse test of PAPER.md:85 on A^{n+1}, folded into barrier S of stage 4
                int any;
                if (MULTI) {
                    wait();
                    any = iflag[par];
                    if (tid == 0) iflag[par ^ 1] = 0;
                } else {
                    any = __syncthreads_or(bad);
                }
                n_done = n + 1;
                if (any && (prm.check_last || n + 1 < prm.nsteps)) collapsed = 1;
                if (collapsed) break;                                     // uniform over the cluster
            } else {
                wait();
            }
        }
        if (collapsed) break;
    }

    // ---- store
    {
        double2 *d0 = reinterpret_cast<double2 *>(prm.U[0] + row + g0);
        double2 *d1 = reinterpret_cast<double2 *>(prm.U[1] + row + g0);
        double2 *d2 = reinterpret_cast<double2 *>(prm.U[2] + row + g0);
#pragma unroll
        for (int p = 0; p < P; p += 2) {
            d0[p / 2] = make_double2(ph[p], ph[p + 1]);
            d1[p / 2] = make_double2(pi[p], pi[p + 1]);
            d2[p / 2] = make_double2(a[p], a[p + 1]);
        }
    }
    if (first) {
        const long long sd = rec->steps_done + n_done;
        rec->steps_done = sd;
        if (collapsed) { rec->collapsed = 1; rec->t_collapse = (double)sd * pb.dt; }
    }
    if (MULTI) cluster.sync();   // no CTA may exit while a neighbour can still write its smem
}

// ------------------------------------------------------------------ configuration table
#define ADSC_RES2_CFG(P_, T_, ACC_)                                                         \
    { "v2P" #P_ "xT" #T_ #ACC_, P_, T_, P_ * T_, ACC_, Res2Layout<P_, T_, ACC_>::bytes, true, \
      { (const void *)k_resident2<P_, T_, ACC_, false>, (const void *)k_resident2<P_, T_, ACC_, true>,     \
        (const void *)k_resident2<P_, T_, ACC_, true>, (const void *)k_resident2<P_, T_, ACC_, true> } }

const ResConfig g_cfgs2[] = {
    ADSC_RES2_CFG(8, 256, true),    // SEG 2048, accumulators in registers
    ADSC_RES2_CFG(8, 256, false),   // SEG 2048, accumulators in shared memory
    ADSC_RES2_CFG(8, 128, false),   // SEG 1024
    ADSC_RES2_CFG(4, 128, false),   // SEG 512
    ADSC_RES2_CFG(4, 64, false),    // SEG 256
    ADSC_RES2_CFG(4, 32, false),    // SEG 128
    ADSC_RES2_CFG(4, 512, false),   // SEG 2048 (experiment: 16 warps)
    ADSC_RES2_CFG(4, 256, false),   // SEG 1024
};
const int n_cfgs2 = sizeof(g_cfgs2) / sizeof(g_cfgs2[0]);

}  // namespace adsc
