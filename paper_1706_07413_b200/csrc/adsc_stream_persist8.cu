// adsc_stream_persist8.cu — persistent streaming kernel, register-blocked version: the chunk logic of
// adsc_stream_persist.cu (stage state of a 7168-point chunk in shared memory, u^n and accumulator through
// global memory, one grid barrier per RK stage, chunk-total suffix scan) with the tile body of the resident
// kernel: 8 contiguous points per thread, 224 threads (7 warps), tiles of 1792 points (4 per chunk),
// state stored [tile][p][thread] so that every warp access is stride-1 (no bank conflicts), the own-point
// fluxes kept in registers and only two flux values per thread edge exchanged through shared memory, TWO
// CTA barriers per tile (scan totals; flux edges) instead of three per 1024 points.
// Equations: eqs (2)-(6); boundary conditions PAPER.md:59-75; algorithm DESIGN.md 1 and 6.
#include <type_traits>

#include "adsc_stream_persist.cuh"
#include "adsc_exp.cuh"

namespace adsc {

// One compiled shape: P contiguous points per thread, T threads, tiles of P*T points, SP_CAP/(P*T) tiles per chunk.
template <int P_, int T_>
struct S8Cfg {
    static constexpr int P = P_, T = T_, NW = T_ / 32, TILE = P_ * T_, TILES = SP_CAP / (P_ * T_), LD = T_ + 2;
    static_assert(TILE * TILES == SP_CAP && T_ % 32 == 0 && P_ >= 4 && P_ % 2 == 0, "tiles must fill the 7168-point chunk");
    static constexpr int o_S = 0;                              // [3][SP_CAP], tile-wise [p][thread]
    static constexpr int o_xH = o_S + 3 * SP_CAP;              // [4][LD]: H at the first two / last two points of each thread
    static constexpr int o_xF = o_xH + 4 * LD;
    static constexpr int o_lo = o_xF + 4 * LD;                 // chunk's lower halo: Phi[3], Pi[3], A[2] at l = -3..-1 / -2..-1
    static constexpr int o_up = o_lo + 8;                      // [2]{Phi[3], Pi[3], A[2]} above the tile (ping-pong by tile)
    static constexpr int o_upf = o_up + 16;                    // [2]{H, H, F, F} at the two points above the tile (ping-pong)
    static constexpr int o_wt = o_upf + 8;                     // [2][8] warp totals (ping-pong by tile)
    static constexpr int o_sw = o_wt + 16;                     // block_sum scratch [8]
    static constexpr int o_gE = o_sw + 8;                      // G_1, G_2, G_{N-2}, G_{N-3}
    static constexpr int o_misc = o_gE + 4;                    // carry, top, flags
    static constexpr int o_eSC = o_misc + 8;                   // -2 sc at every tile boundary -3..+2
    static constexpr int o_eT = o_eSC + 6 * (TILES + 1);       // tan^2 x likewise
    static constexpr int n_doubles = o_eT + 6 * (TILES + 1);
    static constexpr size_t bytes = (size_t)n_doubles * sizeof(double);
    // position of chunk-local index l (0 <= l < SP_CAP) inside a state array
    __device__ static __forceinline__ int pos(int l)
    {
        const int tile = l / TILE, r = l - tile * TILE;
        return tile * TILE + (r % P) * T + (r / P);
    }
};

template <int NW>
__device__ __forceinline__ double s8_block_sum(double v, double *sw)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    __syncthreads();
    if (lane == 0) sw[warp] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) t += sw[w];
    return t;
}

template <int P_, int T_>
__global__ void __launch_bounds__(T_, 1) k_stream_persist8(const __grid_constant__ SPParams prm)
{
    using L = S8Cfg<P_, T_>;
    constexpr int P = L::P, T = L::T, NW = L::NW, LD = L::LD, S8_TILE = L::TILE;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) double smem[];
    double *S = smem + L::o_S, *xH = smem + L::o_xH, *xF = smem + L::o_xF, *lo = smem + L::o_lo;
    double *up = smem + L::o_up, *upf = smem + L::o_upf, *wt = smem + L::o_wt, *sw = smem + L::o_sw;
    double *gE = smem + L::o_gE, *misc = smem + L::o_misc, *eSC = smem + L::o_eSC, *eT = smem + L::o_eT;

    const Problem &pb = prm.pb;
    const SPConsts &K = prm.k;
    const int NS = K.ns, LS = K.ns - 1;      // Runge-Kutta stages (4; 3 or 2 for the rules of reading R25), last stage
    const int N = pb.N, G = prm.G, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, col = tid + 1;
    const int gi = blockIdx.x / G, c = blockIdx.x - gi * G;
    if (gi >= prm.groups) return;
    const int ci0 = c * prm.Lc;                         // first grid index of the chunk
    const int cn = min(prm.Lc, N - ci0);                // points in the chunk (>= 8 by construction)
    const int ntile = (cn + S8_TILE - 1) / S8_TILE;
    const bool owns_top = (ci0 <= N - 2) && (N - 2 < ci0 + cn);     // chunk holding i = N-2
    unsigned long long *cnt = prm.counter + gi;
    double *mb = prm.mbox + (size_t)gi * 2 * G * SP_MBOX;
    unsigned long long epoch = 0;
    const double *__restrict__ tSC = prm.tb.sc;
    const double *__restrict__ tT = prm.tb.T;
    const double *__restrict__ tC = prm.tb.C;
    auto Sg = [&](int v, int l) -> double & { return S[v * SP_CAP + L::pos(l)]; };     // 0 <= l < cn

    // value of field v at chunk-local index l for the edge threads of a tile: below the chunk from `lo`, at and
    // above the tile end from `upb` (the tile above already holds the new stage state), else from the state array
    auto ldv = [&](int v, int l, int tend, const double *upb) -> double {
        if (l < 0) return (v == 2) ? (l >= -2 ? lo[8 + l] : 0.0) : (l >= -3 ? lo[3 * v + 3 + l] : 0.0);
        if (l >= tend) {
            const int k = l - tend;
            if (v == 2) return (k < 2) ? upb[6 + k] : 0.0;
            return (k < 3) ? upb[3 * v + k] : 0.0;
        }
        return Sg(v, l);
    };

    // coefficient tables around every tile boundary of the chunk (used by the two edge threads of a tile)
    if (tid < 6 * (ntile + 1)) {
        const int bd = tid / 6, k = tid - 6 * bd;
        const int j = min(max(ci0 + min(bd * S8_TILE, cn) - 3 + k, -HAL), N - 1 + HAL);
        eSC[tid] = -2.0 * tSC[j]; eT[tid] = tT[j];
    }
    __syncthreads();

    for (int b = gi; b < pb.B; b += prm.groups) {
        MemberRec *rec = prm.rec + b;
        if (rec->collapsed || prm.nsteps <= 0) continue;             // uniform over the group
        const size_t row = (size_t)b * pb.NP;

        // ---- load the chunk; f' total of the initial state
        double facc = 0.0;
        for (int l = tid; l < cn; l += T) {
            const int i = ci0 + l;
            const double p = prm.U[0][row + i], q = prm.U[1][row + i];
            Sg(0, l) = p; Sg(1, l) = q; Sg(2, l) = prm.U[2][row + i];
            if (i <= N - 2) {
                const double f = (-2.0 * tSC[i]) * fma(p, p, q * q);
                facc += f;
                if (i == N - 2) misc[1] = f * (1.0 / 12.0);          // top term of the telescoped rule
            }
        }
        int bad = 0, collapsed = 0;
        long long n = 0;
        unsigned stage_ctr = 0;

        for (;;) {
            for (int s = 0; s < NS; ++s, ++stage_ctr) {
                const int par = (int)(stage_ctr & 1u);
                double *mine = mb + ((size_t)par * G + c) * SP_MBOX;
                // ---- publish: chunk total (+ top), collapse flag, state edges
                double tot = s8_block_sum<NW>(facc, sw);
                if (owns_top) tot += misc[1];
                if (tid == 0) { mine[0] = tot; mine[1] = bad ? 1.0 : 0.0; }
                if (tid < 3) {
                    mine[2 + tid] = Sg(0, tid);           mine[5 + tid] = Sg(1, tid);
                    mine[10 + tid] = Sg(0, cn - 3 + tid); mine[13 + tid] = Sg(1, cn - 3 + tid);
                }
                if (tid < 2) { mine[8 + tid] = Sg(2, tid); mine[16 + tid] = Sg(2, cn - 2 + tid); }
                group_barrier(cnt, (++epoch) * (unsigned long long)G);

                // ---- gather: totals of the chunks above, flags, neighbour edges / parity ghosts
                const double *all = mb + (size_t)par * G * SP_MBOX;
                if (tid < 32) {
                    double cs = 0.0, fl = 0.0;
                    for (int cc = tid; cc < G; cc += 32) {
                        const double t = ld_cg(all + (size_t)cc * SP_MBOX), f = ld_cg(all + (size_t)cc * SP_MBOX + 1);
                        if (cc > c) cs += t;
                        fl += f;
                    }
#pragma unroll
                    for (int d = 16; d >= 1; d >>= 1) {
                        cs += __shfl_xor_sync(FULL, cs, d);
                        fl += __shfl_xor_sync(FULL, fl, d);
                    }
                    if (tid == 0) { misc[0] = cs + (owns_top ? misc[1] : 0.0); misc[2] = fl; }
                } else if (tid < 35) {
                    const int k = tid - 32;                              // 0..2
                    // lower halo: lo[k] = Phi, lo[3+k] = Pi at l = -3+k; lo[6+k] = A at l = -2+k
                    if (c > 0) {
                        const double *below = all + (size_t)(c - 1) * SP_MBOX;
                        lo[k] = ld_cg(below + 10 + k); lo[3 + k] = ld_cg(below + 13 + k);
                        if (k < 2) lo[6 + k] = ld_cg(below + 16 + k);
                    } else {                                             // x = 0: Phi odd, Pi and A even (R2)
                        lo[2 - k] = -Sg(0, 1 + k); lo[5 - k] = Sg(1, 1 + k);
                        if (k < 2) lo[7 - k] = Sg(2, 1 + k);
                    }
                    double *upt = up + 8 * ((ntile - 1) & 1);             // buffer of the chunk's top tile
                    if (c < G - 1) {
                        const double *above = all + (size_t)(c + 1) * SP_MBOX;
                        upt[k] = ld_cg(above + 2 + k); upt[3 + k] = ld_cg(above + 5 + k);
                        if (k < 2) upt[6 + k] = ld_cg(above + 8 + k);
                    } else {                                             // x = pi/2: Phi even, Pi odd (R3)
                        const int lN = N - 1 - ci0;
                        upt[k] = Sg(0, lN - 1 - k); upt[3 + k] = -Sg(1, lN - 1 - k);
                        if (k < 2) upt[6 + k] = Sg(2, lN - 1 - k);
                    }
                }
                __syncthreads();
                if (s == 0) {
                    // a6: collapse test of PAPER.md:85 on the state after n steps (flags of every chunk)
                    if (n > 0 && misc[2] != 0.0) { collapsed = 1; break; }
                    if (n == prm.nsteps) break;                          // final flag round only
                }
                double carry = misc[0];
                facc = 0.0; bad = 0;
                const double a_next = K.a_next[s], b_w = K.b_w[s];

                // ---- tiles, from high x to low x
                double m2n[P + 2];                                        // -2 sc at l0-1 .. l0+P of the coming tile
#pragma unroll
                for (int q = 0; q < P + 2; ++q)
                    m2n[q] = -2.0 * tSC[min(ci0 + (ntile - 1) * S8_TILE + P * tid + q - 1, N - 1)];
                // The tile body is compiled twice: EDGE = true is general (ragged tiles, the tiles at x = 0 and x = pi/2);
                // EDGE = false is for full tiles at least 8 points away from both ends of the grid, where every mask
                // and end-of-domain test below is a compile-time constant and disappears.
                auto tile_body = [&](auto edge_c, const int tt) {
                    constexpr bool EDGE = decltype(edge_c)::value;
                    const int tl0 = tt * S8_TILE;
                    const int tend = EDGE ? min(tl0 + S8_TILE, cn) : tl0 + S8_TILE;
                    const int l0 = tl0 + P * tid;
                    const int i0 = ci0 + l0;                              // global index of my first point
                    const bool any = EDGE ? (l0 < tend) : true;
                    const int nact = (tend - tl0 + P - 1) / P;            // threads that own a point of this tile
                    const bool last_thr = (tid == nact - 1);
                    const bool tile_hi_is_domain_end = EDGE && (ci0 + tend == N);   // the tile holds i = N-1
                    const double *upb = up + 8 * (tt & 1);                // old values above this tile
                    const double *Sb = S + tl0 + tid;                     // (p = 0, my column) of this tile

                    // stage state: u[r] at l0 - 3 + r (r = 0..13): three halo points per side and my eight
                    double uP[P + 6], uQ[P + 6], a[P];
                    if (tid >= 1 && l0 + P + 3 <= tend) {                 // neighbours are columns tid-1, tid+1 of this tile
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            uP[k] = Sb[(P - 3 + k) * T - 1];             uQ[k] = Sb[SP_CAP + (P - 3 + k) * T - 1];
                            uP[P + 3 + k] = Sb[k * T + 1];               uQ[P + 3 + k] = Sb[SP_CAP + k * T + 1];
                        }
#pragma unroll
                        for (int p = 0; p < P; ++p) { uP[3 + p] = Sb[p * T]; uQ[3 + p] = Sb[SP_CAP + p * T]; a[p] = Sb[2 * SP_CAP + p * T]; }
                    } else {
#pragma unroll
                        for (int r = 0; r < P + 6; ++r) { uP[r] = ldv(0, l0 - 3 + r, tend, upb); uQ[r] = ldv(1, l0 - 3 + r, tend, upb); }
#pragma unroll
                        for (int p = 0; p < P; ++p) a[p] = ldv(2, l0 + p, tend, upb);
                    }
                    // old values of this tile's three lowest points: the upper halo of the next (lower) tile
                    if (tid == 0) {
                        double *upn = up + 8 * ((tt & 1) ^ 1);
                        upn[0] = uP[3]; upn[1] = uP[4]; upn[2] = uP[5];
                        upn[3] = uQ[3]; upn[4] = uQ[4]; upn[5] = uQ[5];
                        upn[6] = a[0];  upn[7] = a[1];
                    }
                    // u^n and accumulator of A: issued now, used after the fluxes (eq (4) is combined before barrier F)
                    double ua[P], aa[P];
                    if (any && s > 0) {
                        const double2 *pa = reinterpret_cast<const double2 *>(prm.ACC[2] + row + i0);
#pragma unroll
                        for (int p = 0; p < P; p += 2) { if (EDGE && i0 + p >= pb.NP) continue; const double2 x = pa[p / 2]; aa[p] = x.x; aa[p + 1] = x.y; }
                        if (s < LS) {
                            const double2 *pu = reinterpret_cast<const double2 *>(prm.U[2] + row + i0);
#pragma unroll
                            for (int p = 0; p < P; p += 2) { if (EDGE && i0 + p >= pb.NP) continue; const double2 x = pu[p / 2]; ua[p] = x.x; ua[p + 1] = x.y; }
                        }
                    }
                    // coefficient tables of my points: -2 sc was fetched during the previous tile
                    double m2sc[P], tT8[P];
                    const double m2m = m2n[0], m2p = m2n[P + 1];
#pragma unroll
                    for (int p = 0; p < P; ++p) { m2sc[p] = m2n[1 + p]; tT8[p] = tT[EDGE ? min(i0 + p, N - 1) : i0 + p]; }

                    // a1: f' = -2 sc (Phi^2 + Pi^2) of my points (zero above i = N-2 and outside the chunk)
                    double fo[P], so[P];
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const bool in = !EDGE || ((l0 + p < cn) && (i0 + p <= N - 2));
                        fo[p] = in ? m2sc[p] * fma(uP[3 + p], uP[3 + p], uQ[3 + p] * uQ[3 + p]) : 0.0;
                    }
                    const double fm = m2m * fma(uP[2], uP[2], uQ[2] * uQ[2]);                                  // f'_{l0-1}
                    const double fp = (!EDGE || i0 + P <= N - 2) ? m2p * fma(uP[P + 3], uP[P + 3], uQ[P + 3] * uQ[P + 3]) : 0.0;
                    so[P - 1] = fo[P - 1];
#pragma unroll
                    for (int p = P - 2; p >= 0; --p) so[p] = so[p + 1] + fo[p];
                    // Kreiss-Oliger sums Q Phi, Q Pi of my points (R6); independent of the scan, they fill its latency
                    double kP[P], kQ[P];
                    auto ko_pt = [&](const int p) {
                        double sP = K.kw[0] * uP[3 + p], sQ = K.kw[0] * uQ[3 + p];
#pragma unroll
                        for (int j = 1; j <= 3; ++j) {
                            sP = fma(K.kw[j], uP[3 + p - j] + uP[3 + p + j], sP);
                            sQ = fma(K.kw[j], uQ[3 + p - j] + uQ[3 + p + j], sQ);
                        }
                        kP[p] = sP; kQ[p] = sQ;
                    };
                    // a2: warp-level suffix scan of the thread totals; warp totals to shared memory
                    double incl = so[0];
#pragma unroll
                    for (int k = 0; k < 5; ++k) {
                        const double o = __shfl_down_sync(FULL, incl, 1 << k);
                        if (k < 3) ko_pt(k);
                        if (lane + (1 << k) < 32) incl += o;
                    }
                    const double excl = incl - so[0];
                    const double wsum = __shfl_sync(FULL, incl, 0);
                    double *wtb = wt + 8 * (tt & 1);
                    if (lane == 0) wtb[warp] = wsum;
#pragma unroll
                    for (int p = 3; p < P; ++p) ko_pt(p);
                    __syncthreads();                                      // barrier S: warp totals visible; scratch of the previous tile free
                    double B = excl + carry, ttot = 0.0;
#pragma unroll
                    for (int w = NW - 1; w >= 0; --w) {
                        const double x = wtb[w];
                        if (w > warp) B += x;
                        ttot += x;
                    }
                    // -delta by the telescoped rule, E = e^{-delta}
                    double nd[P], E[P];
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const double f_lo = (p == 0) ? fm : fo[p - 1];
                        const double f_hi = (p == P - 1) ? fp : fo[p + 1];
                        const double s2 = (p + 2 < P) ? so[p + 2] + B : ((p + 2 == P) ? B : B - fp);
                        double loc = K.c25 * f_hi;
                        loc = fma(K.c12, fo[p], loc);
                        loc = fma(-K.c1, f_lo, loc);
                        nd[p] = fma(K.hh, s2, loc);
                    }
                    exp3_near<P>(nd, E);
                    // a3: fluxes of my points
                    double H[P], F[P], kA[P], G1 = 0.0, G2 = 0.0, Gl1 = 0.0, Gl2 = 0.0;
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const double AE = a[p] * E[p];
                        const double Gv = AE * uP[3 + p];
                        H[p] = AE * uQ[3 + p];
                        F[p] = tT8[p] * Gv;
                        kA[p] = (m2sc[p] * a[p]) * (Gv * uQ[3 + p]);                 // eq (4)
                        if (p == 1) G1 = Gv;
                        if (p == 2) G2 = Gv;
                        if (p == P - 1) Gl1 = Gv;
                        if (p == P - 2) Gl2 = Gv;
                        if (EDGE && i0 + p == N - 2) gE[2] = Gv;
                        if (EDGE && i0 + p == N - 3) gE[3] = Gv;
                    }
                    // flux edges of every thread: rows 0, 1 = first two points, rows 2, 3 = last two
                    xH[0 * LD + col] = H[0]; xH[1 * LD + col] = H[1]; xH[2 * LD + col] = H[P - 2]; xH[3 * LD + col] = H[P - 1];
                    xF[0 * LD + col] = F[0]; xF[1 * LD + col] = F[1]; xF[2 * LD + col] = F[P - 2]; xF[3 * LD + col] = F[P - 1];
                    if (tid == 0) {
                        // fluxes at the two points below the tile (column 0, rows 2, 3); at x = 0 the reader mirrors
                        double h1 = 0.0, h2 = 0.0, f1v = 0.0, f2v = 0.0, g1 = 0.0, g2 = 0.0;
                        if (!EDGE || i0 != 0) {
                            const double f1 = fm;                                                          // f'_{l0-1}
                            const double f2 = eSC[6 * tt + 1] * fma(uP[1], uP[1], uQ[1] * uQ[1]);          // f'_{l0-2}
                            const double f3 = eSC[6 * tt] * fma(uP[0], uP[0], uQ[0] * uQ[0]);              // f'_{l0-3}
                            double l1 = K.c25 * fo[0]; l1 = fma(K.c12, f1, l1); l1 = fma(-K.c1, f2, l1);
                            double l2 = K.c25 * f1;    l2 = fma(K.c12, f2, l2); l2 = fma(-K.c1, f3, l2);
                            const double e1 = exp3_ref(fma(K.hh, so[1] + B, l1));
                            const double e2 = exp3_ref(fma(K.hh, so[0] + B, l2));
                            const double ae1 = ldv(2, l0 - 1, tend, upb) * e1, ae2 = ldv(2, l0 - 2, tend, upb) * e2;
                            g1 = ae1 * uP[2]; g2 = ae2 * uP[1];
                            h1 = ae1 * uQ[2]; h2 = ae2 * uQ[1];
                            f1v = eT[6 * tt + 2] * g1; f2v = eT[6 * tt + 1] * g2;
                            xH[3 * LD] = h1; xH[2 * LD] = h2; xF[3 * LD] = f1v; xF[2 * LD] = f2v;
                            if (EDGE && i0 - 1 == N - 2) gE[2] = g1;
                            if (EDGE && i0 - 1 == N - 3) gE[3] = g1;
                            if (EDGE && i0 - 2 == N - 3) gE[3] = g2;
                        }
                        // my first two fluxes are the upper halo of the next (lower) tile
                        double *ufn = upf + 4 * ((tt & 1) ^ 1);
                        if (EDGE && i0 == N - 1) {   // H = 0 at x = pi/2, F by the limit of R5, then mirrored (R3)
                            ufn[0] = 0.0; ufn[1] = -h1; ufn[2] = (16.0 * g1 - g2) * K.inv12h2; ufn[3] = f1v;
                        } else { ufn[0] = H[0]; ufn[1] = H[1]; ufn[2] = F[0]; ufn[3] = F[1]; }
                    }
                    // fluxes at the two points above the tile (column tid+2, rows 0, 1) by the tile's last thread:
                    // from the tile above; for the chunk's top tile from the neighbour chunk's edge values; at
                    // x = pi/2 the reader applies the parity rule itself
                    if (last_thr && !tile_hi_is_domain_end) {
                        double hh0, hh1, ff0, ff1;
                        if (tt < ntile - 1) {
                            const double *uf = upf + 4 * (tt & 1);
                            hh0 = uf[0]; hh1 = uf[1]; ff0 = uf[2]; ff1 = uf[3];
                        } else {
                            const int ie = ci0 + tend;                   // < N-1 here (the top chunk never takes this path)
                            const double f1 = (!EDGE || ie + 1 <= N - 2) ? eSC[6 * (tt + 1) + 4] * fma(uP[P + 4], uP[P + 4], uQ[P + 4] * uQ[P + 4]) : 0.0;
                            const double f2 = (!EDGE || ie + 2 <= N - 2) ? eSC[6 * (tt + 1) + 5] * fma(uP[P + 5], uP[P + 5], uQ[P + 5] * uQ[P + 5]) : 0.0;
                            double l0v = K.c25 * f1; l0v = fma(K.c12, fp, l0v); l0v = fma(-K.c1, fo[P - 1], l0v);
                            double l1v = K.c25 * f2; l1v = fma(K.c12, f1, l1v); l1v = fma(-K.c1, fp, l1v);
                            const double e0 = exp3_ref(fma(K.hh, B - fp - f1, l0v));
                            const double e1 = exp3_ref(fma(K.hh, B - fp - f1 - f2, l1v));
                            const double ae0 = upb[6] * e0, ae1 = upb[7] * e1;
                            const double g0 = ae0 * uP[P + 3], g1 = ae1 * uP[P + 4];
                            hh0 = ae0 * uQ[P + 3]; hh1 = ae1 * uQ[P + 4];
                            ff0 = eT[6 * (tt + 1) + 3] * g0; ff1 = eT[6 * (tt + 1) + 4] * g1;
                            if (EDGE && ie == N - 3) gE[3] = g0;
                            if (EDGE && ie == N - 2) gE[2] = g0;
                            if (EDGE && ie + 1 == N - 3) gE[3] = g1;
                            if (EDGE && ie + 1 == N - 2) gE[2] = g1;
                        }
                        xH[0 * LD + col + 1] = hh0; xH[1 * LD + col + 1] = hh1;
                        xF[0 * LD + col + 1] = ff0; xF[1 * LD + col + 1] = ff1;
                    }
                    // global operands of the second half, issued before the barrier: cot^2 x, u^n and the accumulator of
                    // Phi and Pi (A is combined right here, in the barrier's shadow: eq (4) needs no neighbour), and
                    // -2 sc of the next tile
                    double tC8[P], un0[P], un1[P], ac0[P], ac1[P], nA[P];
#pragma unroll
                    for (int p = 0; p < P; ++p) tC8[p] = tC[EDGE ? min(i0 + p, N - 1) : i0 + p];
#pragma unroll
                    for (int q = 0; q < P + 2; ++q) m2n[q] = -2.0 * tSC[max(i0 + q - 1 - S8_TILE, -1)];
                    if (any) {
                        if (s > 0) {
                            const double2 *p0 = reinterpret_cast<const double2 *>(prm.ACC[0] + row + i0);
                            const double2 *p1 = reinterpret_cast<const double2 *>(prm.ACC[1] + row + i0);
#pragma unroll
                            for (int p = 0; p < P; p += 2) {
                                if (EDGE && i0 + p >= pb.NP) continue;           // (rows are padded to a multiple of 4 only)
                                const double2 x = p0[p / 2], y = p1[p / 2];
                                ac0[p] = x.x; ac0[p + 1] = x.y; ac1[p] = y.x; ac1[p + 1] = y.y;
                            }
                            if (s < LS) {
                                const double2 *q0 = reinterpret_cast<const double2 *>(prm.U[0] + row + i0);
                                const double2 *q1 = reinterpret_cast<const double2 *>(prm.U[1] + row + i0);
#pragma unroll
                                for (int p = 0; p < P; p += 2) {
                                    if (EDGE && i0 + p >= pb.NP) continue;
                                    const double2 x = q0[p / 2], y = q1[p / 2];
                                    un0[p] = x.x; un0[p + 1] = x.y; un1[p] = y.x; un1[p + 1] = y.y;
                                }
                            }
                        }
                        // a4/a5 for A
#pragma unroll
                        for (int p = 0; p < P; ++p) {
                            const int i = i0 + p;
                            const double kAv = (EDGE && (i == 0 || i >= N - 1)) ? 0.0 : kA[p];   // eqs (8), (11)
                            if (s == 0) { aa[p] = fma(b_w, kAv, a[p]); nA[p] = fma(a_next, kAv, a[p]); }
                            else if (s < LS) { aa[p] = fma(b_w, kAv, aa[p]); nA[p] = fma(a_next, kAv, ua[p]); }
                            else {
                                nA[p] = fma(b_w, kAv, aa[p]);
                                if ((!EDGE || (i <= N - 1 && l0 + p < cn)) && !(nA[p] >= K.thr)) bad = 1;   // a6
                            }
                            if (EDGE && i > N - 1) { nA[p] = 0.0; aa[p] = 0.0; }
                        }
                        if (s < LS) {
                            double2 *pa = reinterpret_cast<double2 *>(prm.ACC[2] + row + i0);
#pragma unroll
                            for (int p = 0; p < P; p += 2) { if (!EDGE || i0 + p < pb.NP) pa[p / 2] = make_double2(aa[p], aa[p + 1]); }
                        } else {
                            double2 *pu = reinterpret_cast<double2 *>(prm.U[2] + row + i0);
#pragma unroll
                            for (int p = 0; p < P; p += 2) { if (!EDGE || i0 + p < pb.NP) pu[p / 2] = make_double2(nA[p], nA[p + 1]); }
                        }
                    }
                    __syncthreads();                                      // barrier F: flux edges visible

                    // a4: centred differences of H, F (window l0-2 .. l0+P+1); parity rules at x = 0 and x = pi/2
                    double Hx[P + 4], Fx[P + 4];
                    Hx[0] = xH[2 * LD + col - 1]; Hx[1] = xH[3 * LD + col - 1];
                    Fx[0] = xF[2 * LD + col - 1]; Fx[1] = xF[3 * LD + col - 1];
                    Hx[P + 2] = xH[0 * LD + col + 1]; Hx[P + 3] = xH[1 * LD + col + 1];
                    Fx[P + 2] = xF[0 * LD + col + 1]; Fx[P + 3] = xF[1 * LD + col + 1];
#pragma unroll
                    for (int p = 0; p < P; ++p) { Hx[2 + p] = H[p]; Fx[2 + p] = F[p]; }
                    if (EDGE && i0 == 0) {                   // x = 0: H even, F odd (R2)
                        Hx[0] = Hx[4]; Hx[1] = Hx[3]; Fx[0] = -Fx[4]; Fx[1] = -Fx[3];
                    }
                    if (EDGE && any && i0 + P + 1 >= N - 1) {   // my window reaches i = N-1
                        const double lim = (16.0 * gE[2] - gE[3]) * K.inv12h2;   // F_{N-1} (R5)
#pragma unroll
                        for (int k = 2; k < P + 4; ++k) {
                            const int j = i0 - 2 + k;
                            if (j == N - 1) { Hx[k] = 0.0; Fx[k] = lim; }
                        }
#pragma unroll
                        for (int k = 4; k < P + 4; ++k) {    // j = N, N+1: H odd, F even about x = pi/2 (R3)
                            const int j = i0 - 2 + k;
                            if (j == N) { Hx[k] = -Hx[k - 2]; Fx[k] = Fx[k - 2]; }
                            if (j == N + 1) { Hx[k] = -Hx[k - 4]; Fx[k] = Fx[k - 4]; }
                        }
                    }
                    double nP[P], nQ[P];
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const int i = i0 + p;
                        const double dH = fma(8.0, Hx[p + 3] - Hx[p + 1], Hx[p] - Hx[p + 4]);
                        const double dF = fma(8.0, Fx[p + 3] - Fx[p + 1], Fx[p] - Fx[p + 4]);
                        double vP = fma(K.d4c, dH, kP[p]);
                        double vQ = fma(tC8[p] * K.d4c, dF, kQ[p]);
                        if (EDGE && i == 0) {                // eq (7); Pi_dot(0) = 3 (A e^{-delta} Phi)'(0) (R4)
                            vP = 0.0;
                            vQ = fma(8.0 * G1 - G2, K.c_org, kQ[p]);
                        }
                        if (EDGE && i >= N - 1) { vP = 0.0; vQ = 0.0; }           // eqs (9), (10)
                        // a5: RK combine
                        if (s == 0) {
                            ac0[p] = fma(b_w, vP, uP[3 + p]); ac1[p] = fma(b_w, vQ, uQ[3 + p]);
                            nP[p] = fma(a_next, vP, uP[3 + p]); nQ[p] = fma(a_next, vQ, uQ[3 + p]);
                        } else if (s < LS) {
                            ac0[p] = fma(b_w, vP, ac0[p]); ac1[p] = fma(b_w, vQ, ac1[p]);
                            nP[p] = fma(a_next, vP, un0[p]); nQ[p] = fma(a_next, vQ, un1[p]);
                        } else {
                            nP[p] = fma(b_w, vP, ac0[p]); nQ[p] = fma(b_w, vQ, ac1[p]);
                        }
                        if (EDGE && i > N - 1) { nP[p] = 0.0; nQ[p] = 0.0; ac0[p] = 0.0; ac1[p] = 0.0; }
                    }
                    if (any) {
                        double *Sw = S + tl0 + tid;
#pragma unroll
                        for (int p = 0; p < P; ++p) {
                            if (!EDGE || l0 + p < cn) {
                                Sw[p * T] = nP[p]; Sw[SP_CAP + p * T] = nQ[p]; Sw[2 * SP_CAP + p * T] = nA[p];
                                if (!EDGE || i0 + p <= N - 2) {   // f' of the new stage state, for the next publish
                                    const double f = m2sc[p] * fma(nP[p], nP[p], nQ[p] * nQ[p]);
                                    facc += f;
                                    if (EDGE && i0 + p == N - 2) misc[1] = f * (1.0 / 12.0);
                                }
                            }
                        }
                        double2 *d0 = reinterpret_cast<double2 *>((s < LS ? prm.ACC[0] : prm.U[0]) + row + i0);
                        double2 *d1 = reinterpret_cast<double2 *>((s < LS ? prm.ACC[1] : prm.U[1]) + row + i0);
#pragma unroll
                        for (int p = 0; p < P; p += 2) {
                            if (EDGE && i0 + p >= pb.NP) continue;
                            if (s < LS) { d0[p / 2] = make_double2(ac0[p], ac0[p + 1]); d1[p / 2] = make_double2(ac1[p], ac1[p + 1]); }
                            else { d0[p / 2] = make_double2(nP[p], nP[p + 1]); d1[p / 2] = make_double2(nQ[p], nQ[p + 1]); }
                        }
                    }
                    carry += ttot;
                };   // tile_body
                for (int tt = ntile - 1; tt >= 0; --tt) {
                    // full tile, 8 points clear of x = 0 and of x = pi/2 (uniform over the CTA)
                    const bool interior = (tt + 1) * S8_TILE <= cn && ci0 + tt * S8_TILE >= 8
                                          && ci0 + (tt + 1) * S8_TILE + 8 <= N - 1;
                    if (interior) tile_body(std::false_type{}, tt);
                    else tile_body(std::true_type{}, tt);
                }   // tiles
                bad = __syncthreads_or(bad);
            }   // stages
            if (collapsed || n == prm.nsteps) break;
            ++n;
            if (n == prm.nsteps && !prm.check_last) break;
        }   // steps

        if (c == 0 && tid == 0) {
            const long long sd = rec->steps_done + n;
            rec->steps_done = sd;
            if (collapsed) { rec->collapsed = 1; rec->t_collapse = (double)sd * pb.dt; }
        }
        __syncthreads();
    }   // members
}

template <int P_, int T_>
static cudaError_t launch_shape(adsc_ctx *c, const SPParams &prm)
{
    using L = S8Cfg<P_, T_>;
    const void *fn = (const void *)k_stream_persist8<P_, T_>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::bytes);
    if (e != cudaSuccess) return e;
    void *args[] = { (void *)&prm };
    return cudaLaunchCooperativeKernel(fn, dim3((unsigned)(c->sp_G * c->sp_groups)), dim3(T_), args, L::bytes, c->stream);
}

// shape 8: 8 points x 224 threads (tiles of 1792); shape 84: 4 points x 256 threads (tiles of 1024)
cudaError_t launch_stream_persist8(adsc_ctx *c, const SPParams &prm)
{
    return c->sp_ppt == 84 ? launch_shape<4, 256>(c, prm) : launch_shape<8, 224>(c, prm);
}

}  // namespace adsc
