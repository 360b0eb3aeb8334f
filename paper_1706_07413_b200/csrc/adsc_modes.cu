// adsc_modes.cu — normal-mode projection diagnostic: "the current numerical solution can
// be decomposed into a spectrum of normal modes".  For the AdS4 modes (R19)
//   e_j = d_j cos^3 x 2F1(-j, 3+j; 3/2; sin^2 x),  d_j = sqrt(16 (j+1)(j+2)/pi),  omega_j = 3 + 2j,
// and j < J:  Pi_j = int Pi e_j tan^2 x dx,  Phi_j = int Phi e_j' tan^2 x dx  (composite Simpson, integrand := 0
// at x = pi/2, as for the mass, R15),  E_j = Pi_j^2 + Phi_j^2 / omega_j^2  (R24; sum_j E_j -> M in the linear limit).
// It is a [J x N] . [N x B] contraction whose left factor is never stored: every thread rebuilds the J mode
// values of its grid points with the three-term Jacobi recurrence, 2F1(-j,3+j;3/2;z) = j!/(3/2)_j P_j^{(1/2,3/2)}(1-2z)
// and dP_j^{(a,b)}/dy = (j+a+b+1)/2 P_{j-1}^{(a+1,b+1)}.  A member is cut into S interleaved slices, one CTA each
// (k_mode_partial), and the slice partials are summed in a fixed order (k_mode_finish); off the per-stage path.
#include <cmath>
#include <mutex>

#include "adsc_internal.cuh"

namespace adsc {

constexpr int MODES_MAX = 32;
constexpr int MODES_THREADS = 256;

struct ModeCoef {
    // P_n = (r1[n] y + r2[n]) P_{n-1} - r3[n] P_{n-2} for the families (1/2,3/2) [0] and (3/2,5/2) [1]
    double r1[2][MODES_MAX], r2[2][MODES_MAX], r3[2][MODES_MAX];
    double p1c[2][2];            // P_1 = p1c[.][0] + p1c[.][1] (y - 1)
    double dn[MODES_MAX];        // d_j j!/(3/2)_j
    double dq[MODES_MAX];        // (j + 3)/2: dP_j/dy = dq[j] Q_{j-1}
    double iom2[MODES_MAX];      // 1/omega_j^2
};

// Partial sums of one slice of a member: CTA (b, sl) takes the points i = sl*256 + tid, + S*256, ... (S = gridDim.y
// slices per member) and leaves sum_i w_i tan^2 x_i Pi_i e_j(x_i) / d'_j and the same for Phi e_j' in
// part[b][sl][{0,1}][j] (d'_j = d_j j!/(3/2)_j is applied by k_mode_finish).  Per point and mode: the two Jacobi
// recurrences (6 FP64 instructions) and 4 for the two projections; the weights that do not depend on j are
// formed once per point.
__global__ void __launch_bounds__(MODES_THREADS)
k_mode_partial(Problem pb, Tables tb, const double *__restrict__ gPhi, const double *__restrict__ gPi,
               const __grid_constant__ ModeCoef mc, int J, double *__restrict__ part)
{
    __shared__ double red[2][MODES_THREADS / 32];
    const int b = blockIdx.x, sl = blockIdx.y, S = gridDim.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = pb.N;
    const double *Phi = gPhi + (size_t)b * pb.NP, *Pi = gPi + (size_t)b * pb.NP;
    double sp[MODES_MAX], sf[MODES_MAX];
#pragma unroll
    for (int j = 0; j < MODES_MAX; ++j) { sp[j] = 0.0; sf[j] = 0.0; }
    for (int i = sl * MODES_THREADS + tid; i < N - 1; i += S * MODES_THREADS) {        // the integrand is 0 at i = N-1
        double s, c;
        sincospi((double)i / (2.0 * (double)(N - 1)), &s, &c);
        const double y = c * c - s * s, c2 = c * c, c3 = c2 * c;
        const double wt = tb.w[i] * tb.T[i];
        const double wp = (wt * Pi[i]) * c3;                     // Pi e_j = d'_j c^3 P_j
        const double wf = wt * Phi[i];
        const double wfa = wf * (-3.0 * c2 * s);                 // Phi e_j' = d'_j (-3 c^2 s P_j - 4 s c^4 dq_j Q_{j-1})
        const double wfb = wf * (-4.0 * s * c * c3);
        double p0 = 1.0, p1 = mc.p1c[0][0] + mc.p1c[0][1] * (y - 1.0);      // P_{j-1}, P_j of (1/2, 3/2) at j = 1
        double q0 = 0.0, q1 = 1.0;                                          // Q_{j-2}, Q_{j-1} of (3/2, 5/2) at j = 1
#pragma unroll
        for (int j = 0; j < MODES_MAX; ++j) {
            if (j < J) {
                double Pj, Qjm1;
                if (j == 0) { Pj = 1.0; Qjm1 = 0.0; }
                else if (j == 1) { Pj = p1; Qjm1 = 1.0; }
                else {
                    const double p2 = fma(fma(mc.r1[0][j], y, mc.r2[0][j]), p1, -mc.r3[0][j] * p0);
                    p0 = p1; p1 = p2; Pj = p2;
                    double q2;                                              // Q_{j-1}: index n = j-1 of family 1
                    if (j == 2) q2 = mc.p1c[1][0] + mc.p1c[1][1] * (y - 1.0);
                    else q2 = fma(fma(mc.r1[1][j - 1], y, mc.r2[1][j - 1]), q1, -mc.r3[1][j - 1] * q0);
                    q0 = q1; q1 = q2; Qjm1 = q2;
                }
                sp[j] = fma(wp, Pj, sp[j]);
                sf[j] = fma(wfa, Pj, fma(wfb * mc.dq[j], Qjm1, sf[j]));
            }
        }
    }
    // CTA reduction, mode by mode (fixed order: deterministic)
    double *dst = part + ((size_t)b * S + sl) * 2 * J;
#pragma unroll 1
    for (int j = 0; j < J; ++j) {
        double a = 0.0, f = 0.0;
#pragma unroll
        for (int k = 0; k < MODES_MAX; ++k) if (k == j) { a = sp[k]; f = sf[k]; }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            a += __shfl_down_sync(0xffffffffu, a, d);
            f += __shfl_down_sync(0xffffffffu, f, d);
        }
        __syncthreads();
        if (lane == 0) { red[0][warp] = a; red[1][warp] = f; }
        __syncthreads();
        if (tid == 0) {
            double A = 0.0, F = 0.0;
            for (int w = 0; w < MODES_THREADS / 32; ++w) { A += red[0][w]; F += red[1][w]; }
            dst[j] = A; dst[J + j] = F;
        }
    }
}

// E_j = Pi_j^2 + Phi_j^2 / omega_j^2 from the slice partials, summed in slice order (deterministic).
__global__ void k_mode_finish(int B, int S, int J, const __grid_constant__ ModeCoef mc, const double *__restrict__ part,
                              double *__restrict__ out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= B * J) return;
    const int b = k / J, j = k - b * J;
    double A = 0.0, F = 0.0;
    for (int sl = 0; sl < S; ++sl) {
        const double *src = part + ((size_t)b * S + sl) * 2 * J;
        A += src[j]; F += src[J + j];
    }
    A *= mc.dn[j]; F *= mc.dn[j];
    out[k] = A * A + F * F * mc.iom2[j];
}

// coefficients of the Jacobi recurrence 2n(n+a+b)(2n+a+b-2) P_n =
//   (2n+a+b-1)[(2n+a+b)(2n+a+b-2) y + a^2 - b^2] P_{n-1} - 2(n+a-1)(n+b-1)(2n+a+b) P_{n-2}
static void fill_coef(ModeCoef &mc)
{
    const double ab[2][2] = { { 0.5, 1.5 }, { 1.5, 2.5 } };
    for (int f = 0; f < 2; ++f) {
        const double a = ab[f][0], b = ab[f][1];
        mc.p1c[f][0] = a + 1.0; mc.p1c[f][1] = 0.5 * (a + b + 2.0);
        for (int n = 0; n < MODES_MAX; ++n) {
            mc.r1[f][n] = mc.r2[f][n] = mc.r3[f][n] = 0.0;
            if (n < 2) continue;
            const double c = 2.0 * n + a + b;
            const double a1 = 2.0 * n * (n + a + b) * (c - 2.0);
            mc.r1[f][n] = (c - 1.0) * c * (c - 2.0) / a1;
            mc.r2[f][n] = (c - 1.0) * (a * a - b * b) / a1;
            mc.r3[f][n] = 2.0 * (n + a - 1.0) * (n + b - 1.0) * c / a1;
        }
    }
    double nrm = 1.0;
    for (int j = 0; j < MODES_MAX; ++j) {
        if (j >= 1) nrm *= (double)j / ((double)j + 0.5);
        mc.dn[j] = std::sqrt(16.0 * (j + 1.0) * (j + 2.0) / 3.14159265358979323846264338327950288) * nrm;
        mc.dq[j] = 0.5 * (j + 3.0);
        const double om = 3.0 + 2.0 * j;
        mc.iom2[j] = 1.0 / (om * om);
    }
}

// d_out: [B][J]; scratch: at least B * S * 2 * J doubles.  Slices per member: enough CTAs for two waves of the
// device when the batch alone does not give them, never fewer than 1024 points per CTA.
int mode_slices(const adsc_ctx *c, int J, size_t scratch_doubles)
{
    const int sms = c->dev_sms > 0 ? c->dev_sms : 148;
    int S = (2 * sms + c->pb.B - 1) / c->pb.B;
    const int smax_pts = (c->pb.N + 1023) / 1024;
    if (S > smax_pts) S = smax_pts;
    const size_t smax_mem = scratch_doubles / ((size_t)c->pb.B * 2 * J);
    if ((size_t)S > smax_mem) S = (int)smax_mem;
    if (S > 65535) S = 65535;
    return S < 1 ? 1 : S;
}

cudaError_t launch_mode_energies(adsc_ctx *c, int J, double *d_out, double *scratch, size_t scratch_doubles)
{
    ModeCoef mc;
    fill_coef(mc);
    const int S = mode_slices(c, J, scratch_doubles);
    k_mode_partial<<<dim3((unsigned)c->pb.B, (unsigned)S), MODES_THREADS, 0, c->stream>>>(c->pb, c->tb, c->ws.U[0], c->ws.U[1],
                                                                                        mc, J, scratch);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int n = c->pb.B * J;
    k_mode_finish<<<(n + 127) / 128, 128, 0, c->stream>>>(c->pb.B, S, J, mc, scratch, d_out);
    c->launches++;
    return cudaGetLastError();
}


// ---------------------------------------------------------------------------------------------------------------------
// adsc_mode_energies_static (include/adsc.h): the same projection for a caller that may not allocate device memory.
//
// The projection above keeps its slice partials in the handle's workspace, i.e. in memory somebody had to allocate.
// This variant needs no handle and no workspace: the caller hands over its own Phi, Pi and the output array, and the
// slice partials live in the file-scope device array below, which is part of the library image (the driver places it
// when the library's code is loaded on a device and it stays there until the process exits).  Nothing on this path
// calls cudaMalloc, cudaFree or a library routine that allocates.
//
// k_mode_partial_static is k_mode_partial with the two table look-ups replaced by the arithmetic k_tables uses for them
// (w_i = m_i h / 3, tan^2 x_i = (s/c)^2), and rows of pitch N instead of NP, so that it can read the caller's arrays as
// they are.  Per point the operations and their order are the same, so for the same number of slices the results are
// bitwise those of adsc_mode_energies.

constexpr size_t STATIC_SCRATCH_DOUBLES = ADSC_STATIC_SCRATCH_BYTES / sizeof(double);

// Scratch for the slice partials, [batch][S][2][J] doubles.  One array per device that loads the library, shared by every
// call on that device.  In host code this name is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) double g_mode_scratch[STATIC_SCRATCH_DOUBLES];

__global__ void __launch_bounds__(MODES_THREADS)
k_mode_partial_static(int N, const double *__restrict__ gPhi, const double *__restrict__ gPi,
                      const __grid_constant__ ModeCoef mc, int J, double *__restrict__ part)
{
    __shared__ double red[2][MODES_THREADS / 32];
    const int b = blockIdx.x, sl = blockIdx.y, S = gridDim.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double *Phi = gPhi + (size_t)b * N, *Pi = gPi + (size_t)b * N;
    const double h = 1.5707963267948966192313216916398 / (double)(N - 1);
    double sp[MODES_MAX], sf[MODES_MAX];
#pragma unroll
    for (int j = 0; j < MODES_MAX; ++j) { sp[j] = 0.0; sf[j] = 0.0; }
    for (int i = sl * MODES_THREADS + tid; i < N - 1; i += S * MODES_THREADS) {        // the integrand is 0 at i = N-1
        double s, c;
        sincospi((double)i / (2.0 * (double)(N - 1)), &s, &c);
        if (i == 0) { s = 0.0; c = 1.0; }
        const double y = c * c - s * s, c2 = c * c, c3 = c2 * c;
        const double t = s / c;
        const double wt = (((i == 0) ? 1.0 : ((i & 1) ? 4.0 : 2.0)) * h / 3.0) * (t * t);   // Simpson weight x tan^2 x_i
        const double wp = (wt * Pi[i]) * c3;
        const double wf = wt * Phi[i];
        const double wfa = wf * (-3.0 * c2 * s);
        const double wfb = wf * (-4.0 * s * c * c3);
        double p0 = 1.0, p1 = mc.p1c[0][0] + mc.p1c[0][1] * (y - 1.0);
        double q0 = 0.0, q1 = 1.0;
#pragma unroll
        for (int j = 0; j < MODES_MAX; ++j) {
            if (j < J) {
                double Pj, Qjm1;
                if (j == 0) { Pj = 1.0; Qjm1 = 0.0; }
                else if (j == 1) { Pj = p1; Qjm1 = 1.0; }
                else {
                    const double p2 = fma(fma(mc.r1[0][j], y, mc.r2[0][j]), p1, -mc.r3[0][j] * p0);
                    p0 = p1; p1 = p2; Pj = p2;
                    double q2;
                    if (j == 2) q2 = mc.p1c[1][0] + mc.p1c[1][1] * (y - 1.0);
                    else q2 = fma(fma(mc.r1[1][j - 1], y, mc.r2[1][j - 1]), q1, -mc.r3[1][j - 1] * q0);
                    q0 = q1; q1 = q2; Qjm1 = q2;
                }
                sp[j] = fma(wp, Pj, sp[j]);
                sf[j] = fma(wfa, Pj, fma(wfb * mc.dq[j], Qjm1, sf[j]));
            }
        }
    }
    double *dst = part + ((size_t)b * S + sl) * 2 * J;
#pragma unroll 1
    for (int j = 0; j < J; ++j) {
        double a = 0.0, f = 0.0;
#pragma unroll
        for (int k = 0; k < MODES_MAX; ++k) if (k == j) { a = sp[k]; f = sf[k]; }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            a += __shfl_down_sync(0xffffffffu, a, d);
            f += __shfl_down_sync(0xffffffffu, f, d);
        }
        __syncthreads();
        if (lane == 0) { red[0][warp] = a; red[1][warp] = f; }
        __syncthreads();
        if (tid == 0) {
            double A = 0.0, F = 0.0;
            for (int w = 0; w < MODES_THREADS / 32; ++w) { A += red[0][w]; F += red[1][w]; }
            dst[j] = A; dst[J + j] = F;
        }
    }
}

// Device address of g_mode_scratch on the current device, looked up once per device (the array is a different piece of
// memory on each GPU).  Host code must not pass `g_mode_scratch` itself to a kernel: on the host that name is a shadow
// variable, and a kernel given its address either faults or, on systems where the GPU can reach host memory, quietly
// works on the wrong bytes.
constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex g_scratch_mutex;
static double *g_scratch_addr[STATIC_MAX_DEVICES];   // zero-initialised: not looked up yet

static cudaError_t static_scratch(double **out, int *sms)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    e = cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_mode_scratch);     // `dev` is current: this is ITS copy of the array
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace adsc

using namespace adsc;

extern "C" int adsc_mode_energies_static(int N, int batch, int J, const double *d_Phi, const double *d_Pi,
                                         double *d_E, void *cuda_stream)
{
    if (N < 9 || (N - 1) % 2 != 0) { set_thread_error("adsc_mode_energies_static: N must be >= 9 and odd"); return ADSC_EINVAL; }
    if (batch < 1) { set_thread_error("adsc_mode_energies_static: batch must be >= 1"); return ADSC_EINVAL; }
    if (J < 1 || J > MODES_MAX || 4 * J > N) { set_thread_error("adsc_mode_energies_static: J must be in 1..32 (and <= N/4)"); return ADSC_EINVAL; }
    if (!d_Phi || !d_Pi || !d_E) { set_thread_error("adsc_mode_energies_static: null pointer"); return ADSC_EINVAL; }
    if (((uintptr_t)d_Phi & 7u) || ((uintptr_t)d_Pi & 7u) || ((uintptr_t)d_E & 7u)) {
        set_thread_error("adsc_mode_energies_static: pointers must be 8-byte aligned"); return ADSC_EINVAL;
    }
    // at least one slice per member must fit: batch * 2 * J doubles
    const size_t per_slice = (size_t)batch * 2 * (size_t)J;
    if (per_slice > STATIC_SCRATCH_DOUBLES) {
        set_thread_error("adsc_mode_energies_static: batch * J = " + std::to_string((size_t)batch * J) + " exceeds the built-in scratch ("
                         + std::to_string(STATIC_SCRATCH_DOUBLES / 2) + " = ADSC_STATIC_SCRATCH_BYTES / 16); split the batch or use adsc_mode_energies");
        return ADSC_EINVAL;
    }
    double *scratch = nullptr;
    int sms = 0;
    cudaError_t e = static_scratch(&scratch, &sms);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        set_thread_error(std::string("adsc_mode_energies_static: built-in scratch: ") + cudaGetErrorString(e));
        return ADSC_ECUDA;
    }
    // slices per member, as mode_slices: two waves of CTAs if the batch alone does not give them, at least 1024 points
    // per CTA, and no more than the scratch holds
    long long S = (2LL * sms + batch - 1) / batch;
    const long long smax_pts = ((long long)N + 1023) / 1024;
    if (S > smax_pts) S = smax_pts;
    const long long smax_mem = (long long)(STATIC_SCRATCH_DOUBLES / per_slice);
    if (S > smax_mem) S = smax_mem;
    if (S > 65535) S = 65535;
    if (S < 1) S = 1;
    ModeCoef mc;
    fill_coef(mc);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // Every slot of the scratch that k_mode_finish reads is written by k_mode_partial_static earlier in this call (all
    // batch * S * 2 * J of them), so nothing left over from the previous call is ever read and nothing needs clearing.
    k_mode_partial_static<<<dim3((unsigned)batch, (unsigned)S), MODES_THREADS, 0, st>>>(N, d_Phi, d_Pi, mc, J, scratch);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        const long long n = (long long)batch * J;
        k_mode_finish<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(batch, (int)S, J, mc, scratch, d_E);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        set_thread_error(std::string("adsc_mode_energies_static: kernel launch: ") + cudaGetErrorString(e));
        return ADSC_ECUDA;
    }
    return ADSC_OK;
}
