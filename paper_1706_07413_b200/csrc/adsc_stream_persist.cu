// adsc_stream_persist.cu — persistent streaming kernel: a member too long for one cluster
// (BASELINE.json configs[3], N = 2^20+1) is cut into G contiguous chunks, one per CTA, one CTA per
// SM, all co-resident (cooperative launch).  A CTA keeps the STAGE state (Phi*, Pi*, A*) of its
// chunk in shared memory across all RK stages and steps; u^n and the RK accumulator stream through
// global memory (L2-resident at this size: 6 arrays x 8.4 MB), 216 B per point per RK4 step.
//
// Per RK stage (equations PAPER.md:43-53 eqs (2)-(6); boundary conditions PAPER.md:59-75):
//   publish   chunk total of f' = -2 sin x cos x (Phi^2 + Pi^2), collapse flag, 3-point state edges
//   barrier   one grid-wide barrier over the G CTAs of the member (the delta integration of eq (6)
//             is what the paper calls "order dependent": here it is a three-level
//             suffix scan, thread / CTA tile / chunk totals)
//   tiles     walking the chunk from high x to low x (the direction of the suffix scan, R8), per tile
//             of 1024 points: f', tile scan, delta by the telescoped rule,
//             E = e^{-delta}, fluxes G, H, F, D4 and Kreiss-Oliger stencils, RK combine, in-place
//             write of the new stage state, running sum of the NEW state's f' for the next stage.
// The discrete algorithm is DESIGN.md section 1; nothing here is shared with oracle/.
#include <type_traits>

#include "adsc_stream_persist.cuh"
#include "adsc_exp.cuh"

namespace adsc {

constexpr int SP_HAL = 4;                          // lower halo slots of the chunk arrays (3 used)

// Shared-memory index map: thread t touches P t + q (P = 2 or 4), a stride of P doubles; one padding
// double per 16 makes those accesses conflict-free (16 consecutive lanes, 16 distinct 8-byte banks).
__host__ __device__ constexpr int sp_pad(int j) { return j + (j >> 4); }

// TILE = points per tile (threads x contiguous points per thread), CAP = points per CTA chunk: 7168 with one CTA
// per SM, 3584 with two.
template <int TILE, int CAP>
struct SPLayout {
    static constexpr int SP_TILES = CAP / TILE;
    static_assert(SP_TILES * TILE == CAP, "tiles must fill the chunk");
    static constexpr int field = sp_pad(CAP + SP_HAL + 4) + 1;      // one chunk array with lower halo
    static constexpr int flux = sp_pad(TILE + 4) + 1;               // tile + 2 halo points per side
    static constexpr int o_S = 0;                                   // [3][field]
    static constexpr int o_H = o_S + 3 * field;
    static constexpr int o_F = o_H + flux;
    static constexpr int o_up = o_F + flux;                         // [2]{upP[3], upQ[3], upA[2]} (ping-pong by tile)
    static constexpr int o_sw = o_up + 16;                          // scan scratch [2][40] (ping-pong)
    static constexpr int o_gE = o_sw + 80;                          // G_1, G_2, G_{N-2}, G_{N-3}
    static constexpr int o_misc = o_gE + 4;                         // carry, top, flags ... [8]
    static constexpr int o_eSC = o_misc + 8;                        // -2 sc at every tile boundary -3..+2
    static constexpr int o_eT = o_eSC + 6 * (SP_TILES + 1);         // tan^2 x likewise
    static constexpr int n_doubles = o_eT + 6 * (SP_TILES + 1);
    static constexpr size_t bytes = (size_t)n_doubles * sizeof(double);
};

// Sum over the CTA (result valid in every thread).  sw: 40 doubles.
template <int T>
__device__ __forceinline__ double block_sum(double v, double *sw)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    __syncthreads();
    if (lane == 0) sw[warp] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < T / 32; ++w) t += sw[w];
    return t;
}

// Exclusive suffix over the threads of the CTA: sum of S over threads above this one; total in `total`.
template <int T>
__device__ __forceinline__ double block_suffix_excl_sp(double S, double *sw, double &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double incl = warp_suffix_incl(S);
    if (lane == 0) sw[warp] = incl;          // the caller alternates between two sw buffers
    __syncthreads();
    double above = 0.0, t = 0.0;
#pragma unroll
    for (int w = 0; w < T / 32; ++w) {
        const double x = sw[w];
        t += x;
        if (w > warp) above += x;
    }
    total = t;
    return incl - S + above;
}

// FIXED: A = 1, delta = 0 held fixed (Table II): no f', no scan, E = 1, eq (4) not evolved, no
// collapse test; the mailboxes then carry only the state edges.
// CTAS: CTAs per SM (1: chunks of up to 7168 points; 2: chunks of up to 3584 points, two independent CTAs per SM).
template <int P, int T, bool FIXED, int CTAS>
__global__ void __launch_bounds__(T, CTAS) k_stream_persist(const __grid_constant__ SPParams prm)
{
    constexpr int SP_TILE = P * T;
    static_assert(P >= 2 && (CTAS == 1 || CTAS == 2), "shape");
    using L = SPLayout<SP_TILE, SP_CAP / CTAS>;
    extern __shared__ __align__(16) double smem[];
    double *S = smem + L::o_S, *sH = smem + L::o_H, *sF = smem + L::o_F, *up = smem + L::o_up;
    double *sw = smem + L::o_sw, *gE = smem + L::o_gE, *misc = smem + L::o_misc;
    double *eSC = smem + L::o_eSC, *eT = smem + L::o_eT;
    auto Sv = [&](int v, int l) -> double & { return S[v * L::field + sp_pad(l + SP_HAL)]; };

    const Problem &pb = prm.pb;
    const SPConsts &K = prm.k;
    const int NS = K.ns, LS = K.ns - 1;      // Runge-Kutta stages (4; 3 or 2 for the rules of reading R25), last stage
    const int N = pb.N, G = prm.G, tid = threadIdx.x;
    const int gi = blockIdx.x / G, c = blockIdx.x - gi * G;
    if (gi >= prm.groups) return;
    const int ci0 = c * prm.Lc;                         // first grid index of the chunk
    const int cn = min(prm.Lc, N - ci0);                // points in the chunk (>= 8 by construction)
    const int ntile = (cn + SP_TILE - 1) / SP_TILE;
    const bool owns_top = (ci0 <= N - 2) && (N - 2 < ci0 + cn);     // chunk holding i = N-2
    unsigned long long *cnt = prm.counter + gi;
    double *mb = prm.mbox + (size_t)gi * 2 * G * SP_MBOX;
    unsigned long long epoch = 0;
    const double *__restrict__ tSC = prm.tb.sc;
    const double *__restrict__ tT = prm.tb.T;
    const double *__restrict__ tC = prm.tb.C;

    // value at local index l of field v, l in [tile start - 3, tend + 3): above the tile end the OLD
    // values live in `up` (the tile above has already been overwritten with the new stage state)
    auto ldv = [&](int v, int l, int tend, const double *upb) -> double {
        if (l < tend) return Sv(v, l);
        const int k = l - tend;
        if (v == 2) return (k < 2) ? upb[6 + k] : 0.0;
        return (k < 3) ? upb[3 * v + k] : 0.0;
    };

    // coefficient tables around every tile boundary of the chunk (used by the two edge threads of a tile)
    if (tid < 6 * (ntile + 1)) {
        const int bd = tid / 6, k = tid - 6 * bd;
        const int j = min(max(ci0 + min(bd * SP_TILE, cn) - 3 + k, -HAL), N - 1 + HAL);
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
            Sv(0, l) = p; Sv(1, l) = q; Sv(2, l) = prm.U[2][row + i];
            if (!FIXED && i <= N - 2) {
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
                double tot = block_sum<T>(facc, sw);
                if (owns_top) tot += misc[1];
                if (tid == 0) { mine[0] = tot; mine[1] = bad ? 1.0 : 0.0; }
                if (tid < 3) {
                    mine[2 + tid] = Sv(0, tid);          mine[5 + tid] = Sv(1, tid);
                    mine[10 + tid] = Sv(0, cn - 3 + tid); mine[13 + tid] = Sv(1, cn - 3 + tid);
                }
                if (tid < 2) { mine[8 + tid] = Sv(2, tid); mine[16 + tid] = Sv(2, cn - 2 + tid); }
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
                        cs += __shfl_xor_sync(0xffffffffu, cs, d);
                        fl += __shfl_xor_sync(0xffffffffu, fl, d);
                    }
                    if (tid == 0) { misc[0] = cs + (owns_top ? misc[1] : 0.0); misc[2] = fl; }
                } else if (tid < 35) {
                    const int k = tid - 32;                              // 0..2
                    if (c > 0) {
                        const double *lo = all + (size_t)(c - 1) * SP_MBOX;
                        Sv(0, -3 + k) = ld_cg(lo + 10 + k); Sv(1, -3 + k) = ld_cg(lo + 13 + k);
                        if (k < 2) Sv(2, -2 + k) = ld_cg(lo + 16 + k);
                    } else {                                             // x = 0: Phi odd, Pi and A even (R2)
                        Sv(0, -1 - k) = -Sv(0, 1 + k); Sv(1, -1 - k) = Sv(1, 1 + k); Sv(2, -1 - k) = Sv(2, 1 + k);
                    }
                    double *upt = up + 8 * ((ntile - 1) & 1);             // buffer of the chunk's top tile
                    if (c < G - 1) {
                        const double *hi = all + (size_t)(c + 1) * SP_MBOX;
                        upt[k] = ld_cg(hi + 2 + k); upt[3 + k] = ld_cg(hi + 5 + k);
                        if (k < 2) upt[6 + k] = ld_cg(hi + 8 + k);
                    } else {                                             // x = pi/2: Phi even, Pi odd (R3)
                        const int lN = N - 1 - ci0;
                        upt[k] = Sv(0, lN - 1 - k); upt[3 + k] = -Sv(1, lN - 1 - k);
                        if (k < 2) upt[6 + k] = Sv(2, lN - 1 - k);
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
                double m2n[P + 2];                                            // -2 sc of my points in the coming tile
#pragma unroll
                for (int q = 0; q < P + 2; ++q) m2n[q] = -2.0 * tSC[min(ci0 + (ntile - 1) * SP_TILE + P * tid + q - 1, N - 1)];
                // The tile body is compiled twice: EDGE = true is general (ragged tiles, the tiles at x = 0 and x = pi/2);
                // EDGE = false is for full tiles at least 8 points away from both ends of the grid, where every mask
                // and end-of-domain test below is a compile-time constant and disappears (2/3 of the instructions
                // of the general body are such integer/predicate work).
                auto tile_body = [&](auto edge_c, const int tt) {
                    constexpr bool EDGE = decltype(edge_c)::value;
                    const int tl0 = tt * SP_TILE;
                    const int tend = EDGE ? min(tl0 + SP_TILE, cn) : tl0 + SP_TILE;
                    const int l0 = tl0 + P * tid;
                    const int i0 = ci0 + l0;                              // global index of my first point
                    const bool any = EDGE ? (l0 < tend) : true;
                    const bool tile_hi_is_domain_end = EDGE && (ci0 + tend == N);   // the tile holds i = N-1
                    const bool last_thr = any && (l0 + P >= tend);   // owner of the tile's last point

                    // stage state: ph[r], pi[r] at l0 - 3 + r (r = 0..P+5), a at l0..l0+P-1
                    const double *upb = up + 8 * (tt & 1);                // old values above this tile
                    double ph[P + 6], pi[P + 6], a[P];
                    if (l0 + P + 3 <= tend) {
#pragma unroll
                        for (int r = 0; r < P + 6; ++r) { ph[r] = Sv(0, l0 - 3 + r); pi[r] = Sv(1, l0 - 3 + r); }
#pragma unroll
                        for (int q = 0; q < P; ++q) a[q] = Sv(2, l0 + q);
                    } else {
#pragma unroll
                        for (int r = 0; r < P + 6; ++r) { ph[r] = ldv(0, l0 - 3 + r, tend, upb); pi[r] = ldv(1, l0 - 3 + r, tend, upb); }
#pragma unroll
                        for (int q = 0; q < P; ++q) a[q] = ldv(2, l0 + q, tend, upb);
                    }
                    // old values of this tile's three lowest points: the upper halo of the next (lower) tile
                    if (tid == 0) {
                        double *upn = up + 8 * ((tt & 1) ^ 1);
                        upn[0] = ph[3]; upn[1] = ph[4]; upn[2] = ph[5];
                        upn[3] = pi[3]; upn[4] = pi[4]; upn[5] = pi[5];
                        upn[6] = a[0];  upn[7] = a[1];
                    }
                    // coefficient tables of my points: -2 sc was fetched during the previous tile
                    double m2sc[P], tT4[P], tC4[P];
                    const double m2m = m2n[0], m2p = m2n[P + 1];          // -2 sc at l0 - 1 and l0 + P
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const int it = EDGE ? min(i0 + q, N - 1) : i0 + q;
                        m2sc[q] = m2n[1 + q]; tT4[q] = tT[it]; tC4[q] = tC[it];
                    }

                    // a1: f' = -2 sc (Phi^2 + Pi^2) of my points (zero above i = N-2 and outside the chunk)
                    double fo[P], so[P];
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const bool in = !EDGE || ((l0 + q < cn) && (i0 + q <= N - 2));
                        fo[q] = (in && !FIXED) ? m2sc[q] * fma(ph[3 + q], ph[3 + q], pi[3 + q] * pi[3 + q]) : 0.0;
                    }
                    const double fm = m2m * fma(ph[2], ph[2], pi[2] * pi[2]);                             // f'_{l0-1}
                    const double fp = (!EDGE || i0 + P <= N - 2) ? m2p * fma(ph[P + 3], ph[P + 3], pi[P + 3] * pi[P + 3]) : 0.0;   // f'_{l0+P}
                    so[P - 1] = fo[P - 1];
#pragma unroll
                    for (int q = P - 2; q >= 0; --q) so[q] = so[q + 1] + fo[q];
                    // a2: tile-level suffix scan; B = sum of f' over all points above my four
                    double ttot;
                    double B = 0.0;
                    if constexpr (FIXED) { ttot = 0.0; __syncthreads(); }     // (the barrier also orders the scratch reuse)
                    else B = block_suffix_excl_sp<T>(so[0], sw + 40 * (tt & 1), ttot) + carry;
                    // -delta by the telescoped rule, E = e^{-delta}
                    double nd[P], E[P];
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const double f_lo = (q == 0) ? fm : fo[q - 1];
                        const double f_hi = (q == P - 1) ? fp : fo[q + 1];
                        const double s2 = (q + 2 < P) ? so[q + 2] + B : ((q + 2 == P) ? B : B - fp);
                        double loc = K.c25 * f_hi;
                        loc = fma(K.c12, fo[q], loc);
                        loc = fma(-K.c1, f_lo, loc);
                        nd[q] = fma(K.hh, s2, loc);
                    }
                    if constexpr (FIXED) {
#pragma unroll
                        for (int q = 0; q < P; ++q) E[q] = 1.0;
                    } else exp3_near<P>(nd, E);
                    // a3: fluxes of my points
                    double Hx[P + 4], Fx[P + 4], Gq[P], kA[P];        // Hx[k], Fx[k] at l0 - 2 + k
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const double AE = a[q] * E[q];
                        const double Gv = AE * ph[3 + q];
                        Gq[q] = Gv;
                        Hx[2 + q] = AE * pi[3 + q];
                        Fx[2 + q] = tT4[q] * Gv;
                        kA[q] = FIXED ? 0.0 : (m2sc[q] * a[q]) * (Gv * pi[3 + q]);   // eq (4)
                        sH[sp_pad(2 + P * tid + q)] = Hx[2 + q];
                        sF[sp_pad(2 + P * tid + q)] = Fx[2 + q];
                        if (EDGE && i0 + q == 1) gE[0] = Gv;
                        if (EDGE && i0 + q == 2) gE[1] = Gv;
                        if (EDGE && i0 + q == N - 2) gE[2] = Gv;
                        if (EDGE && i0 + q == N - 3) gE[3] = Gv;
                    }
                    // fluxes at the two points below the tile (thread 0) ...
                    if (tid == 0) {
                        if (!EDGE || i0 != 0) {              // (at x = 0 the reader applies the parity rule)
                            const double f1 = fm;                                                             // f'_{l0-1}
                            const double f2 = eSC[6 * tt + 1] * fma(ph[1], ph[1], pi[1] * pi[1]);             // f'_{l0-2}
                            const double f3 = eSC[6 * tt] * fma(ph[0], ph[0], pi[0] * pi[0]);                 // f'_{l0-3}
                            double l1 = K.c25 * fo[0]; l1 = fma(K.c12, f1, l1); l1 = fma(-K.c1, f2, l1);
                            double l2 = K.c25 * f1;    l2 = fma(K.c12, f2, l2); l2 = fma(-K.c1, f3, l2);
                            const double e1 = FIXED ? 1.0 : exp3_ref(fma(K.hh, so[1] + B, l1));
                            const double e2 = FIXED ? 1.0 : exp3_ref(fma(K.hh, so[0] + B, l2));
                            const double ae1 = Sv(2, l0 - 1) * e1, ae2 = Sv(2, l0 - 2) * e2;
                            const double g1 = ae1 * ph[2], g2 = ae2 * ph[1];
                            sH[sp_pad(1)] = ae1 * pi[2]; sH[sp_pad(0)] = ae2 * pi[1];
                            sF[sp_pad(1)] = eT[6 * tt + 2] * g1; sF[sp_pad(0)] = eT[6 * tt + 1] * g2;
                            if (EDGE && i0 - 1 == N - 2) gE[2] = g1;
                            if (EDGE && i0 - 1 == N - 3) gE[3] = g1;
                            if (EDGE && i0 - 2 == N - 3) gE[3] = g2;
                        }
                    }
                    // ... and at the two points above it (owner of the tile's last point), unless the tile
                    // ends at x = pi/2, where readers apply the parity rule themselves
                    if (last_thr && !tile_hi_is_domain_end) {
                        const int le = tend - tl0 + 2;                   // scratch slot of local index tend
                        const int ie = ci0 + tend;                       // its global index (<= N-1)
                        if (EDGE && ie == N - 1) {           // H = 0 there; F by the limit of R5; then mirrored
                            sH[sp_pad(le)] = 0.0;            sF[sp_pad(le)] = (16.0 * Gq[P - 1] - Gq[P - 2]) * K.inv12h2;
                            sH[sp_pad(le + 1)] = -Hx[P + 1]; sF[sp_pad(le + 1)] = Fx[P + 1];
                        } else {
                            const double f1 = (!EDGE || ie + 1 <= N - 2) ? eSC[6 * (tt + 1) + 4] * fma(ph[P + 4], ph[P + 4], pi[P + 4] * pi[P + 4]) : 0.0;
                            const double f2 = (!EDGE || ie + 2 <= N - 2) ? eSC[6 * (tt + 1) + 5] * fma(ph[P + 5], ph[P + 5], pi[P + 5] * pi[P + 5]) : 0.0;
                            double l0v = K.c25 * f1; l0v = fma(K.c12, fp, l0v); l0v = fma(-K.c1, fo[P - 1], l0v);
                            double l1v = K.c25 * f2; l1v = fma(K.c12, f1, l1v); l1v = fma(-K.c1, fp, l1v);
                            const double e0 = FIXED ? 1.0 : exp3_ref(fma(K.hh, B - fp - f1, l0v));
                            const double e1 = FIXED ? 1.0 : exp3_ref(fma(K.hh, B - fp - f1 - f2, l1v));
                            const double ae0 = upb[6] * e0, ae1 = upb[7] * e1;
                            const double g0 = ae0 * ph[P + 3], g1 = ae1 * ph[P + 4];
                            sH[sp_pad(le)] = ae0 * pi[P + 3]; sH[sp_pad(le + 1)] = ae1 * pi[P + 4];
                            sF[sp_pad(le)] = eT[6 * (tt + 1) + 3] * g0; sF[sp_pad(le + 1)] = eT[6 * (tt + 1) + 4] * g1;
                            if (EDGE && ie == N - 3) gE[3] = g0;
                            if (EDGE && ie == N - 2) gE[2] = g0;
                            if (EDGE && ie + 1 == N - 3) gE[3] = g1;
                            if (EDGE && ie + 1 == N - 2) gE[2] = g1;
                        }
                    }
                    // global operands of the second half (cot^2/(12h), u^n, accumulator) and -2 sc of the next
                    // tile: issued before the barrier so that their latency overlaps it and the stencils
                    double un[3][P], acc[3][P];
#pragma unroll
                    for (int q = 0; q < P + 2; ++q) m2n[q] = -2.0 * tSC[max(i0 + q - 1 - SP_TILE, -1)];
                    if (any && s > 0) {
#pragma unroll
                        for (int v = 0; v < 3; ++v) {
                            const double2 *pa = reinterpret_cast<const double2 *>(prm.ACC[v] + row + i0);
#pragma unroll
                            for (int q = 0; q < P; q += 2) { const double2 x = pa[q / 2]; acc[v][q] = x.x; acc[v][q + 1] = x.y; }
                            if (s < LS) {
                                const double2 *pu = reinterpret_cast<const double2 *>(prm.U[v] + row + i0);
#pragma unroll
                                for (int q = 0; q < P; q += 2) { const double2 y = pu[q / 2]; un[v][q] = y.x; un[v][q + 1] = y.y; }
                            }
                        }
                    }
                    __syncthreads();

                    // a4: centred differences of H, F (neighbours from the scratch; parity rule at x = pi/2)
                    {
                        const int sb = P * tid;                          // scratch slot of local index l0 - 2
                        Hx[0] = sH[sp_pad(sb)];             Hx[1] = sH[sp_pad(sb + 1)];
                        Fx[0] = sF[sp_pad(sb)];             Fx[1] = sF[sp_pad(sb + 1)];
                        Hx[P + 2] = sH[sp_pad(sb + P + 2)]; Hx[P + 3] = sH[sp_pad(sb + P + 3)];
                        Fx[P + 2] = sF[sp_pad(sb + P + 2)]; Fx[P + 3] = sF[sp_pad(sb + P + 3)];
                        if (EDGE && i0 == 0) {               // x = 0: H even, F odd (R2)
                            Hx[0] = Hx[4]; Hx[1] = Hx[3]; Fx[0] = -Fx[4]; Fx[1] = -Fx[3];
                        }
                        if (EDGE && any && i0 + P + 1 >= N - 1) {    // my window l0-2 .. l0+P+1 reaches i = N-1
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
                    }
                    double nP[P], nQ[P], nA[P];
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const int i = i0 + q;
                        const double dH = fma(8.0, Hx[q + 3] - Hx[q + 1], Hx[q] - Hx[q + 4]);
                        const double dF = fma(8.0, Fx[q + 3] - Fx[q + 1], Fx[q] - Fx[q + 4]);
                        double qP = K.kw[0] * ph[3 + q], qQ = K.kw[0] * pi[3 + q];        // Kreiss-Oliger (R6)
#pragma unroll
                        for (int j = 1; j <= 3; ++j) {
                            qP = fma(K.kw[j], ph[3 + q - j] + ph[3 + q + j], qP);
                            qQ = fma(K.kw[j], pi[3 + q - j] + pi[3 + q + j], qQ);
                        }
                        double kP = fma(K.d4c, dH, qP);
                        double kQ = fma(tC4[q] * K.d4c, dF, qQ);
                        double kAv = kA[q];
                        if (EDGE && i == 0) {                // eqs (7), (8); Pi_dot(0) = 3 (A e^{-delta} Phi)'(0) (R4)
                            kP = 0.0; kAv = 0.0;
                            kQ = fma(8.0 * gE[0] - gE[1], K.c_org, qQ);
                        }
                        if (EDGE && i >= N - 1) { kP = 0.0; kQ = 0.0; kAv = 0.0; }   // eqs (9)-(11)
                        // a5: RK combine
                        if (s == 0) {
                            const double u0 = ph[3 + q], u1 = pi[3 + q], u2 = a[q];
                            acc[0][q] = fma(b_w, kP, u0); acc[1][q] = fma(b_w, kQ, u1); acc[2][q] = fma(b_w, kAv, u2);
                            nP[q] = fma(a_next, kP, u0);  nQ[q] = fma(a_next, kQ, u1);  nA[q] = fma(a_next, kAv, u2);
                        } else if (s < LS) {
                            acc[0][q] = fma(b_w, kP, acc[0][q]); acc[1][q] = fma(b_w, kQ, acc[1][q]); acc[2][q] = fma(b_w, kAv, acc[2][q]);
                            nP[q] = fma(a_next, kP, un[0][q]);   nQ[q] = fma(a_next, kQ, un[1][q]);   nA[q] = fma(a_next, kAv, un[2][q]);
                        } else {
                            nP[q] = fma(b_w, kP, acc[0][q]); nQ[q] = fma(b_w, kQ, acc[1][q]); nA[q] = fma(b_w, kAv, acc[2][q]);
                            if (!FIXED && (!EDGE || (i <= N - 1 && l0 + q < cn)) && !(nA[q] >= K.thr)) bad = 1;   // a6
                        }
                        if (EDGE && i > N - 1) { nP[q] = 0.0; nQ[q] = 0.0; nA[q] = 0.0; acc[0][q] = 0.0; acc[1][q] = 0.0; acc[2][q] = 0.0; }
                    }
                    if (any) {
#pragma unroll
                        for (int q = 0; q < P; ++q) {
                            if (!EDGE || l0 + q < cn) {
                                Sv(0, l0 + q) = nP[q]; Sv(1, l0 + q) = nQ[q]; Sv(2, l0 + q) = nA[q];
                                if (!FIXED && (!EDGE || i0 + q <= N - 2)) {   // f' of the new stage state, for the next publish
                                    const double f = m2sc[q] * fma(nP[q], nP[q], nQ[q] * nQ[q]);
                                    facc += f;
                                    if (EDGE && i0 + q == N - 2) misc[1] = f * (1.0 / 12.0);
                                }
                            }
                        }
                        if (s < LS) {
#pragma unroll
                            for (int v = 0; v < 3; ++v) {
                                double2 *pa = reinterpret_cast<double2 *>(prm.ACC[v] + row + i0);
#pragma unroll
                                for (int q = 0; q < P; q += 2) pa[q / 2] = make_double2(acc[v][q], acc[v][q + 1]);
                            }
                        } else {
                            double2 *p0 = reinterpret_cast<double2 *>(prm.U[0] + row + i0);
                            double2 *p1 = reinterpret_cast<double2 *>(prm.U[1] + row + i0);
                            double2 *p2 = reinterpret_cast<double2 *>(prm.U[2] + row + i0);
#pragma unroll
                            for (int q = 0; q < P; q += 2) {
                                p0[q / 2] = make_double2(nP[q], nP[q + 1]);
                                p1[q / 2] = make_double2(nQ[q], nQ[q + 1]);
                                p2[q / 2] = make_double2(nA[q], nA[q + 1]);
                            }
                        }
                    }
                    carry += ttot;
                };   // tile_body
                for (int tt = ntile - 1; tt >= 0; --tt) {
                    // full tile, 8 points clear of x = 0 and of x = pi/2 (uniform over the CTA)
                    const bool interior = (tt + 1) * SP_TILE <= cn && ci0 + tt * SP_TILE >= 8
                                          && ci0 + (tt + 1) * SP_TILE + 8 <= N - 1;
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


// ------------------------------------------------------------------ host side
// Chunks per member G and concurrent members: every CTA of a member must be co-resident (one CTA per
// SM), a chunk holds at most SP_CAP points and at least one tile's worth (so the last chunk keeps >= 8).
bool stream_persist_select(adsc_ctx *c)
{
    c->sp_ok = false;
    if (c->dev_sms <= 0) return false;
    if (c->pb.fixed_bg && (c->sp_ppt == 8 || c->sp_ppt == 84 || c->sp_ppt == 42)) c->sp_ppt = 4;   // no fixed-background build
    if (c->sp_ppt != 2 && c->sp_ppt != 4 && c->sp_ppt != 8 && c->sp_ppt != 84 && c->sp_ppt != 42) c->sp_ppt = 4;
    const int ctas = (c->sp_ppt == 42) ? 2 : 1;                        // CTAs per SM
    const int cap = SP_CAP / ctas, tile = (c->sp_ppt == 42) ? 512 : 1024;
    const int N = c->pb.N, sms = c->dev_sms * ctas;                    // co-resident CTAs
    const int gmin = (N + cap - 1) / cap;
    if (gmin > sms) return false;
    const int per_member = sms / (c->pb.B < sms ? c->pb.B : sms);      // CTAs a member can have
    int G = per_member;
    const int gmax = (N + tile - 1) / tile;
    if (G > gmax) G = gmax;
    if (G < gmin) G = gmin;
    const int al = (c->sp_ppt == 8) ? 8 : 4;                 // chunks start on a thread boundary
    int Lc = ((N + G - 1) / G + al - 1) / al * al;
    G = (N + Lc - 1) / Lc;
    if (Lc > cap || (G > 1 && N - (G - 1) * Lc < 8)) return false;
    int groups = sms / G;
    if (groups > c->pb.B) groups = c->pb.B;
    if (groups < 1 || (size_t)groups * G > SP_MAX_CTAS) return false;
    c->sp_G = G; c->sp_Lc = Lc; c->sp_groups = groups; c->sp_ok = true;
    return true;
}

cudaError_t launch_stream_persist(adsc_ctx *c, long long nsteps, int check_last)
{
    const void *fn;
    int threads = 256;
    size_t smem = SPLayout<1024, SP_CAP>::bytes;
    if (c->pb.fixed_bg) {
        if (c->sp_ppt == 2) { fn = (const void *)k_stream_persist<2, 512, true, 1>; threads = 512; }
        else fn = (const void *)k_stream_persist<4, 256, true, 1>;
    } else if (c->sp_ppt == 42) {
        fn = (const void *)k_stream_persist<4, 128, false, 2>; threads = 128; smem = SPLayout<512, SP_CAP / 2>::bytes;
    } else if (c->sp_ppt == 2) { fn = (const void *)k_stream_persist<2, 512, false, 1>; threads = 512; }
    else fn = (const void *)k_stream_persist<4, 256, false, 1>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(c->ws.sp_counter, 0, sizeof(unsigned long long) * SP_MAX_CTAS, c->stream);
    if (e != cudaSuccess) return e;
    SPParams prm;
    prm.pb = c->pb; prm.tb = c->tb;
    for (int v = 0; v < 3; ++v) { prm.U[v] = c->ws.U[v]; prm.ACC[v] = c->ws.ACC[v]; }
    prm.rec = c->ws.rec; prm.mbox = c->ws.sp_mbox; prm.counter = c->ws.sp_counter;
    prm.nsteps = nsteps; prm.check_last = check_last;
    prm.G = c->sp_G; prm.groups = c->sp_groups; prm.Lc = c->sp_Lc;
    {
        const double h = c->pb.h, dt = c->pb.dt, koc = c->pb.ko_eps / (64.0 * h);
        SPConsts &k = prm.k;
        k.d4c = 1.0 / (12.0 * h);
        k.kw[0] = -20.0 * koc; k.kw[1] = 15.0 * koc; k.kw[2] = -6.0 * koc; k.kw[3] = koc;
        k.hh = 0.5 * h; k.c25 = 25.0 * h / 48.0; k.c12 = 0.25 * h; k.c1 = h / 48.0;
        k.inv12h2 = 1.0 / (12.0 * h * h); k.c_org = 1.0 / (2.0 * h);
        rk_tableau(c->rk_order, dt, k.a_next, k.b_w);
        k.ns = c->rk_order;
        k.thr = c->pb.thr;
    }
    if (c->sp_ppt == 8 || c->sp_ppt == 84) {
        e = launch_stream_persist8(c, prm);
        c->launches++;
        return e;
    }
    void *args[] = { (void *)&prm };
    e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)(c->sp_G * c->sp_groups)), dim3((unsigned)threads), args,
                                    smem, c->stream);
    c->launches++;
    return e;
}

}  // namespace adsc
