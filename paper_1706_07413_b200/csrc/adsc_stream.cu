// adsc_stream.cu — streaming (global-memory) RK4 stage kernels: any N, any batch.
// Used when a member does not fit on chip (BASELINE.json configs[3], N = 2^20+1) and as
// the general fallback.  Per RK stage:
//   k_stream_I      a1 + tile part of a2: f, I, tile-local suffix sums, tile totals
//   k_stream_carry  a2 across tiles: exclusive suffix of the tile totals (deterministic)
//   k_stream_rhs    a3 + a4 + a5 (+ a6 at stage 4): delta, fluxes, stencils, KO, RK combine
// Equations: eqs (2)-(6); BCs PAPER.md:59-75 eqs (7)-(12).
#include "adsc_internal.cuh"

namespace adsc {

constexpr int PPT = GEN_TILE / GEN_THREADS;   // 4

__device__ __forceinline__ double tile_suffix_excl(double S, double *sw, double &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = GEN_THREADS >> 5;
    double incl = warp_suffix_incl(S);
    if (lane == 0) sw[warp] = incl;
    __syncthreads();
    double v = (lane < nw) ? sw[lane] : 0.0;
    double vi = warp_suffix_incl(v);                       // every warp redundantly
    double above = __shfl_sync(0xffffffffu, vi - v, warp); // sum over warps above mine
    total = __shfl_sync(0xffffffffu, vi, 0);
    return incl - S + above;
}

// a1 (+ tile-local a2).  Grid (ntiles, B).
__global__ void __launch_bounds__(GEN_THREADS)
k_stream_I(Problem pb, Tables tb, const double *__restrict__ gPhi, const double *__restrict__ gPi,
           double *__restrict__ gdl, double *__restrict__ gtot, const MemberRec *__restrict__ rec, int ntiles)
{
    __shared__ double sw[32];
    const int b = blockIdx.y, tile = blockIdx.x, tid = threadIdx.x;
    if (rec[b].collapsed) return;
    const int N = pb.N;
    const double *Phi = gPhi + (size_t)b * pb.NP, *Pi = gPi + (size_t)b * pb.NP;
    const double c13 = 13.0 * pb.h / 24.0, c1 = pb.h / 24.0;
    const int i0 = tile * GEN_TILE + PPT * tid;
    double f[PPT + 3];
#pragma unroll
    for (int q = 0; q < PPT + 3; ++q) {
        const int j = i0 - 1 + q;
        double v = 0.0;
        if (j <= N + 1) {
            double ph = ld_ghost(Phi, j, N, -1, +1), pi = ld_ghost(Pi, j, N, +1, -1);
            v = tb.sc[j] * (ph * ph + pi * pi);
        }
        f[q] = v;
    }
    double loc[PPT];
#pragma unroll
    for (int q = PPT - 1; q >= 0; --q) {
        double I = (i0 + q <= N - 2) ? (c13 * (f[q + 1] + f[q + 2]) - c1 * (f[q] + f[q + 3])) : 0.0;
        loc[q] = (q == PPT - 1) ? I : loc[q + 1] + I;
    }
    double total;
    const double excl = tile_suffix_excl(loc[0], sw, total);
    double *dl = gdl + (size_t)b * pb.NP;
#pragma unroll
    for (int q = 0; q < PPT; ++q)
        if (i0 + q <= N - 1) dl[i0 + q] = loc[q] + excl;   // dl[N-1] = 0
    if (tid == 0) gtot[(size_t)b * ntiles + tile] = total;
}

// a2 across tiles.  Grid B; exclusive suffix of tot over tiles, walked from the top.
__global__ void __launch_bounds__(GEN_THREADS)
k_stream_carry(const double *__restrict__ gtot, double *__restrict__ gcarry,
               const MemberRec *__restrict__ rec, int ntiles)
{
    __shared__ double sw[32];
    const int b = blockIdx.x, tid = threadIdx.x;
    if (rec[b].collapsed) return;
    const double *tot = gtot + (size_t)b * ntiles;
    double *carry = gcarry + (size_t)b * ntiles;
    double run = 0.0;
    const int nch = (ntiles + GEN_THREADS - 1) / GEN_THREADS;
    for (int ch = nch - 1; ch >= 0; --ch) {
        const int t = ch * GEN_THREADS + tid;
        const double v = (t < ntiles) ? tot[t] : 0.0;
        double total;
        const double excl = tile_suffix_excl(v, sw, total);
        if (t < ntiles) carry[t] = excl + run;
        run += total;
        __syncthreads();
    }
}

struct Flux { double G, H, F; };

// G = A e^{-delta} Phi, H = A e^{-delta} Pi, F = tan^2 x G at a physical index m in [0, N-2].
__device__ __forceinline__ Flux flux_phys(const Problem &pb, const Tables &tb, const double *Phi,
                                          const double *Pi, const double *A, const double *dl,
                                          const double *carry, int m)
{
    // fixed background: delta = 0 is not integrated, e^{-delta} = 1
    const double AE = pb.fixed_bg ? A[m] : A[m] * exp(-(dl[m] + carry[m / GEN_TILE]));
    Flux r;
    r.G = AE * Phi[m];
    r.H = AE * Pi[m];
    r.F = tb.T[m] * r.G;
    return r;
}

// Flux at any logical index j in [-2, N+1] with the parities G(-,+) H(+,-) F(-,+) and the
// boundary limit F_{N-1} = (16 G_{N-2} - G_{N-3})/(12 h^2) (R5).
__device__ Flux flux_at(const Problem &pb, const Tables &tb, const double *Phi, const double *Pi,
                        const double *A, const double *dl, const double *carry, int j)
{
    const int N = pb.N;
    double sG = 1.0, sH = 1.0;
    int m = j;
    if (j < 0) { m = -j; sG = -1.0; sH = 1.0; }
    else if (j > N - 1) { m = 2 * (N - 1) - j; sG = 1.0; sH = -1.0; }
    Flux r;
    if (m == N - 1) {
        Flux a = flux_phys(pb, tb, Phi, Pi, A, dl, carry, N - 2);
        Flux c = flux_phys(pb, tb, Phi, Pi, A, dl, carry, N - 3);
        r.G = 0.0; r.H = 0.0;
        r.F = (16.0 * a.G - c.G) / (12.0 * pb.h * pb.h);
    } else {
        r = flux_phys(pb, tb, Phi, Pi, A, dl, carry, m);
        r.G *= sG; r.H *= sH; r.F *= sG;
    }
    return r;
}

struct StageIO {
    const double *in[3];    // stage state u*
    const double *un[3];    // u^n
    double *acc[3];         // u^n + dt/6 * (running sum)
    double *out[3];         // next stage state (or u^{n+1} at stage 4)
};

// a3-a6.  Grid (ntiles, B).
__global__ void __launch_bounds__(GEN_THREADS)
k_stream_rhs(Problem pb, Tables tb, StageIO io, const double *__restrict__ gdl,
             const double *__restrict__ gcarry, MemberRec *rec, int ntiles, int stage, int last_stage,
             double a_next, double b_w)
{
    __shared__ double sG[GEN_TILE + 2 * HAL], sH[GEN_TILE + 2 * HAL], sF[GEN_TILE + 2 * HAL];
    const int b = blockIdx.y, tile = blockIdx.x, tid = threadIdx.x;
    if (rec[b].collapsed) return;
    const int N = pb.N;
    const size_t row = (size_t)b * pb.NP;
    const double *Phi = io.in[0] + row, *Pi = io.in[1] + row, *A = io.in[2] + row;
    const double *dl = gdl + row, *carry = gcarry + (size_t)b * ntiles;
    const int base = tile * GEN_TILE;
    const int i0 = base + PPT * tid;

    double a_own[PPT], pi_own[PPT];
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
        const int j = i0 + q;
        Flux fx; fx.G = fx.H = fx.F = 0.0;
        a_own[q] = 1.0; pi_own[q] = 0.0;
        if (j <= N + 1) {
            fx = flux_at(pb, tb, Phi, Pi, A, dl, carry, j);
            if (j <= N - 1) { a_own[q] = A[j]; pi_own[q] = Pi[j]; }
        }
        sG[HAL + PPT * tid + q] = fx.G; sH[HAL + PPT * tid + q] = fx.H; sF[HAL + PPT * tid + q] = fx.F;
    }
    if (tid < 4) {
        const int j = (tid < 2) ? (base - 2 + tid) : (base + GEN_TILE + tid - 2);
        Flux fx; fx.G = fx.H = fx.F = 0.0;
        if (j >= -2 && j <= N + 1) fx = flux_at(pb, tb, Phi, Pi, A, dl, carry, j);
        const int s = (tid < 2) ? (HAL - 2 + tid) : (HAL + GEN_TILE + tid - 2);
        sG[s] = fx.G; sH[s] = fx.H; sF[s] = fx.F;
    }
    __syncthreads();

    const double d4c = 1.0 / (12.0 * pb.h), koc = pb.ko_eps / (64.0 * pb.h);
    int bad = 0;
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
        const int i = i0 + q;
        if (i > N - 1) continue;
        const int s = HAL + PPT * tid + q;
        double ph[7], pq[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            ph[k] = ld_ghost(Phi, i - 3 + k, N, -1, +1);
            pq[k] = ld_ghost(Pi, i - 3 + k, N, +1, -1);
        }
        const double qPhi = koc * (ph[0] - 6.0 * ph[1] + 15.0 * ph[2] - 20.0 * ph[3] + 15.0 * ph[4] - 6.0 * ph[5] + ph[6]);
        const double qPi = koc * (pq[0] - 6.0 * pq[1] + 15.0 * pq[2] - 20.0 * pq[3] + 15.0 * pq[4] - 6.0 * pq[5] + pq[6]);
        double k[3];
        k[0] = d4c * (sH[s - 2] - 8.0 * sH[s - 1] + 8.0 * sH[s + 1] - sH[s + 2]) + qPhi;
        if (i == 0)
            k[1] = 3.0 * d4c * (sG[s - 2] - 8.0 * sG[s - 1] + 8.0 * sG[s + 1] - sG[s + 2]) + qPi;
        else
            k[1] = tb.C[i] * (d4c * (sF[s - 2] - 8.0 * sF[s - 1] + 8.0 * sF[s + 1] - sF[s + 2])) + qPi;
        k[2] = pb.fixed_bg ? 0.0 : -2.0 * tb.sc[i] * a_own[q] * sG[s] * pi_own[q];
        if (i == 0) { k[0] = 0.0; k[2] = 0.0; }
        if (i == N - 1) { k[0] = 0.0; k[1] = 0.0; k[2] = 0.0; }
#pragma unroll
        for (int v = 0; v < 3; ++v) {
            const size_t g = row + i;
            const double base_un = io.un[v][g];
            const double accv = (stage == 0) ? base_un : io.acc[v][g];
            const double accn = accv + b_w * k[v];
            if (stage < last_stage) {
                io.acc[v][g] = accn;
                io.out[v][g] = base_un + a_next * k[v];
            } else {
                io.out[v][g] = accn;
                if (v == 2 && !pb.fixed_bg && !(accn >= pb.thr)) bad = 1;
            }
        }
    }
    if (stage == last_stage) {
        if (__syncthreads_or(bad) && tid == 0) atomicOr(&rec[b].bad, 1);
    }
}

cudaError_t launch_stream_step(adsc_ctx *c)
{
    const int nt = c->lay.ntiles;
    dim3 grid(nt, c->pb.B);
    Workspace &w = c->ws;
    double a_next[4], b_w[4];
    rk_tableau(c->rk_order, c->pb.dt, a_next, b_w);
    const int ns = c->rk_order, last = ns - 1;
    for (int s = 0; s < ns; ++s) {
        // stage states ping-pong between Ua and Ub; the first stage reads, the last one writes, the state U
        double *const *in = (s == 0) ? w.U : ((s & 1) ? w.Ua : w.Ub);
        double *const *out = (s == last) ? w.U : ((s & 1) ? w.Ub : w.Ua);
        if (!c->pb.fixed_bg) {
            k_stream_I<<<grid, GEN_THREADS, 0, c->stream>>>(c->pb, c->tb, in[0], in[1], w.dl, w.tot, w.rec, nt);
            k_stream_carry<<<c->pb.B, GEN_THREADS, 0, c->stream>>>(w.tot, w.carry, w.rec, nt);
            c->launches += 2;
        }
        StageIO io;
        for (int v = 0; v < 3; ++v) { io.in[v] = in[v]; io.un[v] = w.U[v]; io.acc[v] = w.ACC[v]; io.out[v] = out[v]; }
        k_stream_rhs<<<grid, GEN_THREADS, 0, c->stream>>>(c->pb, c->tb, io, w.dl, w.carry, w.rec, nt, s, last, a_next[s], b_w[s]);
        c->launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace adsc
