// adsc_solve_tiled.cu — the constraint integrations of eqs (5), (6) and the
// diagnostics of PAPER.md:83-85 for LONG members (streaming layouts, N >= 32768): the same
// arithmetic as k_solve (adsc_setup.cu), but a member is cut into tiles of 1024 points that run on
// different CTAs, with a tile-total carry pass between the local scans (reduce-then-scan, so the
// result is deterministic).  k_solve walks one member with ONE CTA, which takes 4.3 ms at
// N = 2^20+1; this path takes six short launches.
//   k_st_delta_local   f, I, tile-local suffix sums of I, tile totals            (eq 6, R7, R8)
//   k_st_carry         exclusive suffix (delta) or prefix (A) of the tile totals
//   k_st_A_local       p = tan^2 x (Phi^2+Pi^2) e^{-delta}, J, tile-local prefix sums, totals (eq 5, R11)
//   k_st_apply         delta_i final; A^c_i = 1 - e^{delta_i} (cos^3/sin)_i P_i; diagnostics partials
//   k_st_reduce        per-member reduction of the partials into the member record
#include "adsc_internal.cuh"

namespace adsc {

constexpr int ST_PPT = GEN_TILE / GEN_THREADS;   // 4

// Exclusive suffix (dir = 0) or prefix (dir = 1) of S over the threads of the CTA; total of all in `total`.
__device__ __forceinline__ double st_block_excl(double S, double *sw, double &total, int dir)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = GEN_THREADS >> 5;
    const double incl = dir ? warp_prefix_incl(S) : warp_suffix_incl(S);
    __syncthreads();
    if (lane == (dir ? 31 : 0)) sw[warp] = incl;
    __syncthreads();
    double other = 0.0, t = 0.0;
#pragma unroll
    for (int w = 0; w < nw; ++w) {
        const double x = sw[w];
        t += x;
        if (dir ? (w < warp) : (w > warp)) other += x;
    }
    total = t;
    return incl - S + other;
}

__global__ void __launch_bounds__(GEN_THREADS)
k_st_delta_local(Problem pb, Tables tb, const double *__restrict__ gPhi, const double *__restrict__ gPi,
                 double *__restrict__ gdl, double *__restrict__ gtot, const MemberRec *__restrict__ rec,
                 int ntiles, int mode)
{
    __shared__ double sw[32];
    const int b = blockIdx.y, tile = blockIdx.x, tid = threadIdx.x;
    if ((mode & SOLVE_ACTIVE_ONLY) && rec[b].collapsed) return;
    const int N = pb.N;
    const double *Phi = gPhi + (size_t)b * pb.NP, *Pi = gPi + (size_t)b * pb.NP;
    const double c13 = 13.0 * pb.h / 24.0, c1 = pb.h / 24.0;
    const int i0 = tile * GEN_TILE + ST_PPT * tid;
    double f[ST_PPT + 3];
#pragma unroll
    for (int q = 0; q < ST_PPT + 3; ++q) {
        const int j = i0 - 1 + q;
        double v = 0.0;
        if (j <= N + 1) {
            const double ph = ld_ghost(Phi, j, N, -1, +1), pi = ld_ghost(Pi, j, N, +1, -1);
            v = tb.sc[j] * (ph * ph + pi * pi);
        }
        f[q] = v;
    }
    double loc[ST_PPT];
#pragma unroll
    for (int q = ST_PPT - 1; q >= 0; --q) {
        const double I = (i0 + q <= N - 2) ? (c13 * (f[q + 1] + f[q + 2]) - c1 * (f[q] + f[q + 3])) : 0.0;
        loc[q] = (q == ST_PPT - 1) ? I : loc[q + 1] + I;
    }
    double total;
    const double excl = st_block_excl(loc[0], sw, total, 0);
    double *dl = gdl + (size_t)b * pb.NP;
#pragma unroll
    for (int q = 0; q < ST_PPT; ++q)
        if (i0 + q <= N - 1) dl[i0 + q] = loc[q] + excl;     // tile-local; dl[N-1] = 0
    if (tid == 0) gtot[(size_t)b * ntiles + tile] = total;
}

// Grid B.  dir = 0: carry[t] = sum of tot over tiles above t; dir = 1: over tiles below t.
__global__ void __launch_bounds__(GEN_THREADS)
k_st_carry(const double *__restrict__ gtot, double *__restrict__ gcarry, const MemberRec *__restrict__ rec,
           int ntiles, int mode, int dir)
{
    __shared__ double sw[32];
    const int b = blockIdx.x, tid = threadIdx.x;
    if ((mode & SOLVE_ACTIVE_ONLY) && rec[b].collapsed) return;
    const double *tot = gtot + (size_t)b * ntiles;
    double *carry = gcarry + (size_t)b * ntiles;
    double run = 0.0;
    const int nch = (ntiles + GEN_THREADS - 1) / GEN_THREADS;
    for (int k = 0; k < nch; ++k) {
        const int ch = dir ? k : nch - 1 - k;
        const int t = ch * GEN_THREADS + tid;
        const double v = (t < ntiles) ? tot[t] : 0.0;
        double total;
        const double excl = st_block_excl(v, sw, total, dir);
        if (t < ntiles) carry[t] = excl + run;
        run += total;
    }
}

__global__ void __launch_bounds__(GEN_THREADS)
k_st_A_local(Problem pb, Tables tb, const double *__restrict__ gPhi, const double *__restrict__ gPi,
             const double *__restrict__ gdl, const double *__restrict__ gcarry, double *__restrict__ gPex,
             double *__restrict__ gtot2, const MemberRec *__restrict__ rec, int ntiles, int mode)
{
    __shared__ double sw[32];
    const int b = blockIdx.y, tile = blockIdx.x, tid = threadIdx.x;
    if ((mode & SOLVE_ACTIVE_ONLY) && rec[b].collapsed) return;
    const int N = pb.N;
    const size_t row = (size_t)b * pb.NP;
    const double *Phi = gPhi + row, *Pi = gPi + row, *dl = gdl + row;
    const double *carry = gcarry + (size_t)b * ntiles;
    const double c13 = 13.0 * pb.h / 24.0, c1 = pb.h / 24.0;
    const int i0 = tile * GEN_TILE + ST_PPT * tid;
    double p[ST_PPT + 3];
#pragma unroll
    for (int q = 0; q < ST_PPT + 3; ++q) {
        const int j = i0 - 1 + q;
        double v = 0.0;
        if (j <= N + 1) {
            double sg;
            const int m = mirror(j, N, +1, +1, sg);            // p is even at both ends
            if (m != N - 1) {
                const double ph = Phi[m], pi = Pi[m];
                const double dj = dl[m] + carry[m / GEN_TILE];
                v = tb.T[m] * (ph * ph + pi * pi) * exp(-dj);
            }
        }
        p[q] = v;
    }
    double loc[ST_PPT];
#pragma unroll
    for (int q = 0; q < ST_PPT; ++q) {
        const double J = (i0 + q <= N - 2) ? (c13 * (p[q + 1] + p[q + 2]) - c1 * (p[q] + p[q + 3])) : 0.0;
        loc[q] = (q == 0) ? J : loc[q - 1] + J;
    }
    double total;
    const double excl = st_block_excl(loc[ST_PPT - 1], sw, total, 1);
    double *Pex = gPex + row;
#pragma unroll
    for (int q = 0; q < ST_PPT; ++q)
        if (i0 + q <= N - 1) Pex[i0 + q] = excl + (q > 0 ? loc[q - 1] : 0.0);   // sum of J below i, inside the tile
    if (tid == 0) gtot2[(size_t)b * ntiles + tile] = total;
}

// part[b][tile][0..5] = mass, resid, min A, argmin (as double), nan flag, bad flag
__global__ void __launch_bounds__(GEN_THREADS)
k_st_apply(Problem pb, Tables tb, const double *__restrict__ gPhi, const double *__restrict__ gPi, double *gA,
           double *gdl, const double *__restrict__ gcarry, double *gAc, const double *__restrict__ gcarry2,
           double *__restrict__ gpart, const MemberRec *__restrict__ rec, int ntiles, int mode)
{
    __shared__ double red[6][GEN_THREADS / 32];
    const int b = blockIdx.y, tile = blockIdx.x, tid = threadIdx.x;
    if ((mode & SOLVE_ACTIVE_ONLY) && rec[b].collapsed) return;
    const int N = pb.N;
    const size_t row = (size_t)b * pb.NP;
    const double cd = gcarry[(size_t)b * ntiles + tile];
    const bool solveA = (mode & (SOLVE_WRITE_A | SOLVE_DIAG)) != 0;
    const double cp = solveA ? gcarry2[(size_t)b * ntiles + tile] : 0.0;
    double t_mass = 0.0, t_res = 0.0, t_min = __longlong_as_double(0x7ff0000000000000LL);
    int t_arg = 0x7fffffff, t_bad = 0, t_nan = 0;
    const int i0 = tile * GEN_TILE + ST_PPT * tid;
#pragma unroll
    for (int q = 0; q < ST_PPT; ++q) {
        const int i = i0 + q;
        if (i > N - 1) continue;
        const double dlt = (i == N - 1) ? 0.0 : gdl[row + i] + cd;
        gdl[row + i] = dlt;                                    // delta final (eq 6, gauge eq 12)
        if (!solveA) continue;
        double a = 1.0;
        if (i >= 1 && i <= N - 2) a = 1.0 - exp(dlt) * tb.c3s[i] * (gAc[row + i] + cp);
        double a_state;
        if (mode & SOLVE_WRITE_A) { gA[row + i] = a; a_state = a; }
        else { gAc[row + i] = a; a_state = gA[row + i]; }
        if (mode & SOLVE_DIAG) {
            const double ph = gPhi[row + i], pi = gPi[row + i];
            if (i < N - 1) t_mass += tb.w[i] * (tb.T[i] * a_state * (ph * ph + pi * pi));
            const double d = fabs(a_state - a);
            if (d != d) t_nan = 1;
            t_res = fmax(t_res, d);
            if (a_state < t_min) { t_min = a_state; t_arg = i; }
        }
        if (!(a_state >= pb.thr)) t_bad = 1;
    }
    if (!solveA) return;
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        t_mass += __shfl_down_sync(0xffffffffu, t_mass, d);
        t_res = fmax(t_res, __shfl_down_sync(0xffffffffu, t_res, d));
        t_nan |= __shfl_down_sync(0xffffffffu, t_nan, d);
        t_bad |= __shfl_down_sync(0xffffffffu, t_bad, d);
        const double om = __shfl_down_sync(0xffffffffu, t_min, d);
        const int oa = __shfl_down_sync(0xffffffffu, t_arg, d);
        if (om < t_min || (om == t_min && oa < t_arg)) { t_min = om; t_arg = oa; }
    }
    if (lane == 0) {
        red[0][warp] = t_mass; red[1][warp] = t_res; red[2][warp] = t_min;
        red[3][warp] = (double)t_arg; red[4][warp] = (double)t_nan; red[5][warp] = (double)t_bad;
    }
    __syncthreads();
    if (tid == 0) {
        double M = 0.0, R = 0.0, mn = red[2][0], ar = red[3][0], nn = 0.0, bd = 0.0;
        for (int w = 0; w < GEN_THREADS / 32; ++w) {
            M += red[0][w]; R = fmax(R, red[1][w]); nn += red[4][w]; bd += red[5][w];
            if (red[2][w] < mn || (red[2][w] == mn && red[3][w] < ar)) { mn = red[2][w]; ar = red[3][w]; }
        }
        double *o = gpart + ((size_t)b * ntiles + tile) * 6;
        o[0] = M; o[1] = R; o[2] = mn; o[3] = ar; o[4] = nn; o[5] = bd;
    }
}

__global__ void __launch_bounds__(GEN_THREADS)
k_st_reduce(const double *__restrict__ gpart, MemberRec *rec, int ntiles, int mode)
{
    __shared__ double red[6][GEN_THREADS / 32];
    const int b = blockIdx.x, tid = threadIdx.x;
    if ((mode & SOLVE_ACTIVE_ONLY) && rec[b].collapsed) return;
    double M = 0.0, R = 0.0, mn = __longlong_as_double(0x7ff0000000000000LL), ar = 2147483647.0, nn = 0.0, bd = 0.0;
    for (int t = tid; t < ntiles; t += GEN_THREADS) {       // fixed assignment and order: deterministic
        const double *o = gpart + ((size_t)b * ntiles + t) * 6;
        M += o[0]; R = fmax(R, o[1]); nn += o[4]; bd += o[5];
        if (o[2] < mn || (o[2] == mn && o[3] < ar)) { mn = o[2]; ar = o[3]; }
    }
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        M += __shfl_down_sync(0xffffffffu, M, d);
        R = fmax(R, __shfl_down_sync(0xffffffffu, R, d));
        nn += __shfl_down_sync(0xffffffffu, nn, d);
        bd += __shfl_down_sync(0xffffffffu, bd, d);
        const double om = __shfl_down_sync(0xffffffffu, mn, d), oa = __shfl_down_sync(0xffffffffu, ar, d);
        if (om < mn || (om == mn && oa < ar)) { mn = om; ar = oa; }
    }
    if (lane == 0) { red[0][warp] = M; red[1][warp] = R; red[2][warp] = mn; red[3][warp] = ar; red[4][warp] = nn; red[5][warp] = bd; }
    __syncthreads();
    if (tid == 0) {
        M = 0.0; R = 0.0; nn = 0.0; bd = 0.0; mn = red[2][0]; ar = red[3][0];
        for (int w = 0; w < GEN_THREADS / 32; ++w) {
            M += red[0][w]; R = fmax(R, red[1][w]); nn += red[4][w]; bd += red[5][w];
            if (red[2][w] < mn || (red[2][w] == mn && red[3][w] < ar)) { mn = red[2][w]; ar = red[3][w]; }
        }
        if (mode & SOLVE_DIAG) {
            rec[b].mass = M;
            rec[b].resid = (nn != 0.0) ? __longlong_as_double(0x7ff8000000000000LL) : R;
            rec[b].min_A = mn;
            rec[b].argmin_A = (ar >= 2147483647.0) ? 0 : (int)ar;
        }
        if (mode & SOLVE_WRITE_A) rec[b].bad = (bd != 0.0) ? 1 : 0;
    }
}

cudaError_t launch_solve_tiled(adsc_ctx *c, int mode)
{
    const int nt = c->lay.ntiles;
    const dim3 grid(nt, c->pb.B);
    Workspace &w = c->ws;
    k_st_delta_local<<<grid, GEN_THREADS, 0, c->stream>>>(c->pb, c->tb, w.U[0], w.U[1], w.dl, w.tot, w.rec, nt, mode);
    k_st_carry<<<c->pb.B, GEN_THREADS, 0, c->stream>>>(w.tot, w.carry, w.rec, nt, mode, 0);
    c->launches += 2;
    const bool solveA = (mode & (SOLVE_WRITE_A | SOLVE_DIAG)) != 0;
    if (solveA) {
        k_st_A_local<<<grid, GEN_THREADS, 0, c->stream>>>(c->pb, c->tb, w.U[0], w.U[1], w.dl, w.carry, w.Ac, w.tot2,
                                                          w.rec, nt, mode);
        k_st_carry<<<c->pb.B, GEN_THREADS, 0, c->stream>>>(w.tot2, w.carry2, w.rec, nt, mode, 1);
        c->launches += 2;
    }
    k_st_apply<<<grid, GEN_THREADS, 0, c->stream>>>(c->pb, c->tb, w.U[0], w.U[1], w.U[2], w.dl, w.carry, w.Ac, w.carry2,
                                                    w.part, w.rec, nt, mode);
    c->launches += 1;
    if (solveA) {
        k_st_reduce<<<c->pb.B, GEN_THREADS, 0, c->stream>>>(w.part, w.rec, nt, mode);
        c->launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace adsc
