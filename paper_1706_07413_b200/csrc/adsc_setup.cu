// adsc_setup.cu — coefficient tables, pack/unpack, the constraint integrations of
// eqs (5),(6) as chunked CTA-wide fp64 scans, and the per-member
// diagnostics of PAPER.md:83-85.  These run at set_initial / diagnostics / get_fields /
// every K_A steps; they are off the per-stage path, so one CTA walks one member.
#include "adsc_internal.cuh"

namespace adsc {

constexpr int SOLVE_THREADS = 512;
constexpr int SOLVE_PPT = 4;
constexpr int SOLVE_CHUNK = SOLVE_THREADS * SOLVE_PPT;

// ------------------------------------------------------------------------------ tables
// x_i = i*h with h = (pi/2)/(N-1): sin/cos via sincospi(i/(2(N-1))) so the argument
// reduction is exact.  Ghost entries carry the mirrored value with the table's parity.
__global__ void k_tables(int N, int NP, double *tab)
{
    const int NT = NP + 2 * HAL;
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= NT) return;
    int j = k - HAL;              // logical index, may be a ghost
    double sg_odd = 1.0;
    int i = j;
    if (i < 0) { i = -i; sg_odd = -1.0; }
    else if (i > N - 1) { i = 2 * (N - 1) - i; sg_odd = -1.0; }
    const bool inside = (j >= 0 && j <= N - 1);
    double s, c;
    sincospi((double)i / (2.0 * (double)(N - 1)), &s, &c);
    if (i == 0) { s = 0.0; c = 1.0; }
    if (i == N - 1) { s = 1.0; c = 0.0; }
    double sc = 0.0, T = 0.0, C = 0.0, c3s = 0.0, w = 0.0;
    if (i <= N - 1 && i >= 0 && j <= N - 1 + HAL) {
        sc = s * c;
        if (i < N - 1) { double t = s / c; T = t * t; }
        if (i >= 1 && i <= N - 2) { double t = c / s; C = t * t; c3s = c * c * c / s; }
        if (inside) {
            const double h = 1.5707963267948966192313216916398 / (double)(N - 1);
            double m = (i == 0 || i == N - 1) ? 1.0 : ((i & 1) ? 4.0 : 2.0);
            w = m * h / 3.0;
        }
    }
    tab[0 * (size_t)NT + k] = sg_odd * sc;
    tab[1 * (size_t)NT + k] = T;
    tab[2 * (size_t)NT + k] = C;
    tab[3 * (size_t)NT + k] = sg_odd * c3s;
    tab[4 * (size_t)NT + k] = w;
}

cudaError_t launch_tables(adsc_ctx *c)
{
    const int NT = c->pb.NP + 2 * HAL;
    k_tables<<<(NT + 255) / 256, 256, 0, c->stream>>>(c->pb.N, c->pb.NP, c->ws.tab);
    c->launches++;
    return cudaGetLastError();
}

// -------------------------------------------------------------------------- pack/unpack
// External rows [B][N] (8-byte aligned) <-> internal rows [B][NP] (32-byte aligned).
// field 0 = Phi (Phi_0 = Phi_{N-1} = 0, eqs 7, 9), 1 = Pi (Pi_{N-1} = 0, eq 10),
// 2 = A (A_0 = A_{N-1} = 1, eqs 8, 11).
__global__ void k_pack(Problem pb, const double *__restrict__ src, double *__restrict__ dst,
                       int field, MemberRec *rec, int init_rec)
{
    const int b = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < pb.NP) {
        double v = 0.0;
        if (i < pb.N) {
            v = src[(size_t)b * pb.N + i];
            if (field == 0 && (i == 0 || i == pb.N - 1)) v = 0.0;
            if (field == 1 && i == pb.N - 1) v = 0.0;
            if (field == 2 && (i == 0 || i == pb.N - 1)) v = 1.0;
        }
        dst[(size_t)b * pb.NP + i] = v;
    }
    if (init_rec && blockIdx.x == 0 && threadIdx.x == 0) {
        MemberRec r;
        r.steps_done = 0; r.t_collapse = __longlong_as_double(0x7ff8000000000000LL);
        r.min_A = 1.0; r.mass = 0.0; r.resid = 0.0; r.argmin_A = 0; r.collapsed = 0; r.bad = 0; r.pad = 0;
        rec[b] = r;
    }
}

cudaError_t launch_pack(adsc_ctx *c, const double *src, int field, bool init_rec)
{
    dim3 grid((c->pb.NP + 255) / 256, c->pb.B);
    k_pack<<<grid, 256, 0, c->stream>>>(c->pb, src, c->ws.U[field], field, c->ws.rec, init_rec ? 1 : 0);
    c->launches++;
    return cudaGetLastError();
}

__global__ void k_unpack(Problem pb, const double *__restrict__ src, double *__restrict__ dst)
{
    const int b = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < pb.N) dst[(size_t)b * pb.N + i] = src[(size_t)b * pb.NP + i];
}

__global__ void k_fill(size_t n, double *__restrict__ dst, double value)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = value;
}

cudaError_t launch_fill(adsc_ctx *c, double *dst_internal, double value)
{
    const size_t n = (size_t)c->pb.B * c->pb.NP;
    k_fill<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, dst_internal, value);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_unpack(adsc_ctx *c, const double *src_internal, double *dst)
{
    dim3 grid((c->pb.N + 255) / 256, c->pb.B);
    k_unpack<<<grid, 256, 0, c->stream>>>(c->pb, src_internal, dst);
    c->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------ block scans
// Exclusive suffix / prefix over the threads of a CTA (<= 32 warps).  sw: 33 doubles.
__device__ __forceinline__ double block_suffix_excl(double S, double *sw, double &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    double incl = warp_suffix_incl(S);
    if (lane == 0) sw[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        double v = (lane < nw) ? sw[lane] : 0.0;
        double vi = warp_suffix_incl(v);
        sw[lane] = vi - v;
        if (lane == 0) sw[32] = vi;
    }
    __syncthreads();
    total = sw[32];
    double r = incl - S + sw[warp];
    __syncthreads();
    return r;
}

__device__ __forceinline__ double block_prefix_excl(double S, double *sw, double &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    double incl = warp_prefix_incl(S);
    if (lane == 31) sw[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        double v = (lane < nw) ? sw[lane] : 0.0;
        double vi = warp_prefix_incl(v);
        sw[lane] = vi - v;
        if (lane == 31) sw[32] = vi;
    }
    __syncthreads();
    total = sw[32];
    double r = incl - S + sw[warp];
    __syncthreads();
    return r;
}

// -------------------------------------------------------------------- constraint solves
// One CTA per member.
//  pass 1 (eq 6, gauge eq 12): f = sc (Phi^2+Pi^2);
//     I_i = (h/24)[13(f_i+f_{i+1}) - (f_{i-1}+f_{i+2})]; delta_i = sum_{k>=i} I_k (suffix scan,
//     chunks walked from x=pi/2 inward with a running carry).
//  pass 2 (eq 5, integrated form, R11): p = tan^2 x (Phi^2+Pi^2) e^{-delta};
//     J_i from p by the same rule; P_i = sum_{k<i} J_k (prefix scan);
//     A_i = 1 - e^{delta_i} (cos^3/sin)_i P_i, A_0 = A_{N-1} = 1.
//  diagnostics: Simpson mass, max|A - A^c|, min A / argmin.
__global__ void __launch_bounds__(SOLVE_THREADS)
k_solve(Problem pb, Tables tb, const double *__restrict__ gPhi, const double *__restrict__ gPi,
        double *gA, double *gdelta, double *gAc, MemberRec *rec, int mode)
{
    __shared__ double sw[33];
    __shared__ double red[3][SOLVE_THREADS / 32];
    __shared__ int redi[2][SOLVE_THREADS / 32];
    const int b = blockIdx.x;
    if ((mode & SOLVE_ACTIVE_ONLY) && rec[b].collapsed) return;
    const int N = pb.N, tid = threadIdx.x;
    const double *Phi = gPhi + (size_t)b * pb.NP, *Pi = gPi + (size_t)b * pb.NP;
    double *A = gA + (size_t)b * pb.NP;
    double *delta = gdelta + (size_t)b * pb.NP;
    double *Ac = gAc + (size_t)b * pb.NP;
    const double c13 = 13.0 * pb.h / 24.0, c1 = pb.h / 24.0;
    const int nI = N - 1;
    const int nch = (nI + SOLVE_CHUNK - 1) / SOLVE_CHUNK;

    // ---- pass 1: delta
    double carry = 0.0;
    if (tid == 0) delta[N - 1] = 0.0;
    for (int ch = nch - 1; ch >= 0; --ch) {
        const int i0 = ch * SOLVE_CHUNK + SOLVE_PPT * tid;
        double f[SOLVE_PPT + 3];
#pragma unroll
        for (int q = 0; q < SOLVE_PPT + 3; ++q) {
            int j = i0 - 1 + q;
            double v = 0.0;
            if (j <= N + 1) {
                double ph = ld_ghost(Phi, j, N, -1, +1), pi = ld_ghost(Pi, j, N, +1, -1);
                v = tb.sc[j] * (ph * ph + pi * pi);
            }
            f[q] = v;
        }
        double loc[SOLVE_PPT];
#pragma unroll
        for (int q = SOLVE_PPT - 1; q >= 0; --q) {
            double I = (i0 + q <= N - 2) ? (c13 * (f[q + 1] + f[q + 2]) - c1 * (f[q] + f[q + 3])) : 0.0;
            loc[q] = (q == SOLVE_PPT - 1) ? I : loc[q + 1] + I;
        }
        double total;
        double excl = block_suffix_excl(loc[0], sw, total);
#pragma unroll
        for (int q = 0; q < SOLVE_PPT; ++q)
            if (i0 + q <= N - 2) delta[i0 + q] = loc[q] + (excl + carry);
        carry += total;
    }
    __syncthreads();
    if (!(mode & (SOLVE_WRITE_A | SOLVE_DIAG))) return;

    // ---- pass 2: A^c, and diagnostics
    double *Aout = (mode & SOLVE_WRITE_A) ? A : Ac;
    double t_mass = 0.0, t_res = 0.0, t_min = __longlong_as_double(0x7ff0000000000000LL);
    int t_arg = 0x7fffffff, t_bad = 0, t_nan = 0;
    carry = 0.0;
    if (tid == 0) { Aout[0] = 1.0; Aout[N - 1] = 1.0; }
    for (int ch = 0; ch < nch; ++ch) {
        const int i0 = ch * SOLVE_CHUNK + SOLVE_PPT * tid;
        double p[SOLVE_PPT + 3], dl0[SOLVE_PPT], s2[SOLVE_PPT];
#pragma unroll
        for (int q = 0; q < SOLVE_PPT + 3; ++q) {
            int j = i0 - 1 + q;
            double v = 0.0, dj = 0.0, ss = 0.0;
            if (j <= N + 1) {
                double sg;
                int m = mirror(j, N, +1, +1, sg);
                if (m != N - 1) {
                    double ph = Phi[m], pi = Pi[m];
                    dj = delta[m];
                    ss = ph * ph + pi * pi;
                    v = tb.T[m] * ss * exp(-dj);
                }
            }
            p[q] = v;
            if (q >= 1 && q <= SOLVE_PPT) { dl0[q - 1] = dj; s2[q - 1] = ss; }
        }
        double loc[SOLVE_PPT];
#pragma unroll
        for (int q = 0; q < SOLVE_PPT; ++q) {
            double J = (i0 + q <= N - 2) ? (c13 * (p[q + 1] + p[q + 2]) - c1 * (p[q] + p[q + 3])) : 0.0;
            loc[q] = (q == 0) ? J : loc[q - 1] + J;
        }
        double total;
        double excl = block_prefix_excl(loc[SOLVE_PPT - 1], sw, total);
#pragma unroll
        for (int q = 0; q < SOLVE_PPT; ++q) {
            const int i = i0 + q;
            if (i <= N - 1) {
                double Pint = (excl + carry) + (q > 0 ? loc[q - 1] : 0.0);
                double a = 1.0;
                if (i >= 1 && i <= N - 2) {
                    a = 1.0 - exp(dl0[q]) * tb.c3s[i] * Pint;
                    Aout[i] = a;
                }
                double a_state = (mode & SOLVE_WRITE_A) ? a : A[i];
                if (mode & SOLVE_DIAG) {
                    if (i < N - 1) t_mass += tb.w[i] * (tb.T[i] * a_state * s2[q]);
                    double d = fabs(a_state - a);
                    if (d != d) t_nan = 1;
                    t_res = fmax(t_res, d);
                    if (a_state < t_min) { t_min = a_state; t_arg = i; }
                }
                if (!(a_state >= pb.thr)) t_bad = 1;
            }
        }
        carry += total;
    }
    // ---- block reductions
    const int lane = tid & 31, warp = tid >> 5;
    const int any_bad = __syncthreads_or(t_bad);
    if (mode & SOLVE_DIAG) {
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            t_mass += __shfl_down_sync(0xffffffffu, t_mass, d);
            t_res = fmax(t_res, __shfl_down_sync(0xffffffffu, t_res, d));
            t_nan |= __shfl_down_sync(0xffffffffu, t_nan, d);
            double om = __shfl_down_sync(0xffffffffu, t_min, d);
            int oa = __shfl_down_sync(0xffffffffu, t_arg, d);
            if (om < t_min || (om == t_min && oa < t_arg)) { t_min = om; t_arg = oa; }
        }
        if (lane == 0) { red[0][warp] = t_mass; red[1][warp] = t_res; red[2][warp] = t_min;
                         redi[0][warp] = t_arg; redi[1][warp] = t_nan; }
        __syncthreads();
        if (tid == 0) {
            double M = 0.0, R = 0.0, mn = red[2][0]; int ar = redi[0][0], nn = 0;
            for (int w = 0; w < SOLVE_THREADS / 32; ++w) {
                M += red[0][w]; R = fmax(R, red[1][w]); nn |= redi[1][w];
                if (red[2][w] < mn || (red[2][w] == mn && redi[0][w] < ar)) { mn = red[2][w]; ar = redi[0][w]; }
            }
            rec[b].mass = M;
            rec[b].resid = nn ? __longlong_as_double(0x7ff8000000000000LL) : R;
            rec[b].min_A = mn; rec[b].argmin_A = (ar == 0x7fffffff) ? 0 : ar;
        }
    }
    if ((mode & SOLVE_WRITE_A) && tid == 0) rec[b].bad = any_bad ? 1 : 0;
}

cudaError_t launch_solve(adsc_ctx *c, int mode)
{
    if (c->path != 2 && c->pb.N >= SOLVE_TILED_MIN_N) return launch_solve_tiled(c, mode);
    k_solve<<<c->pb.B, SOLVE_THREADS, 0, c->stream>>>(c->pb, c->tb, c->ws.U[0], c->ws.U[1], c->ws.U[2],
                                                     c->ws.dl, c->ws.Ac, c->ws.rec, mode);
    c->launches++;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------- finalize
// Per member, after a step: count it, apply the collapse test result.
__global__ void k_finalize(Problem pb, MemberRec *rec, int inc_steps)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= pb.B) return;
    MemberRec r = rec[b];
    if (!r.collapsed) {
        if (inc_steps) r.steps_done += 1;
        if (r.bad) { r.collapsed = 1; r.t_collapse = (double)r.steps_done * pb.dt; }
    }
    r.bad = 0;
    rec[b] = r;
}

cudaError_t launch_finalize(adsc_ctx *c, int inc_steps)
{
    k_finalize<<<(c->pb.B + 127) / 128, 128, 0, c->stream>>>(c->pb, c->ws.rec, inc_steps);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace adsc
