// adsc_resident3.cuh — the resident Runge-Kutta kernel: one ensemble member per CTA (or per cluster of CL CTAs),
// the whole state on chip across all RK stages and steps.  (Instantiated in adsc_resident3_{a,b,c,d}.cu; host side in
// adsc_resident.cu.)
//
// Arithmetic per stage: telescoped delta rule, two synchronisation points per RK
// stage, one full exp per thread and short relative polynomials for the other points.  Design decisions
// (against the two earlier generations of this kernel, both removed: "v1" with three cluster barriers per stage, "v2"
// with the same arithmetic as this one but cluster barriers), and why:
//   * Synchronisation is point-to-point.  Every sync point is an mbarrier in each CTA's shared memory:
//     one elected lane per warp arrives on it (split arrive / wait, so the independent arithmetic
//     placed between them overlaps the skew between warps also inside ONE CTA), and data for other
//     CTAs of the cluster travels by st.async straight into the consumer's shared memory, completing
//     transaction bytes on the consumer's mbarrier.  No barrier.cluster and no cluster-scope fence in the
//     loop: the v2 cluster kernel spent 0.75 stall cycles per issued instruction in `membar` and
//     ~490 clk per cluster barrier.
//   * All scalars derived from h, dt, eps_KO sit in the kernel parameter bank (ResConsts) and the exp
//     coefficients in __constant__ memory, so fp64 instructions take them as c[][] operands: v2
//     re-materialised ~70 64-bit immediates per thread and stage with IMAD.MOV (8.7 % of all
//     instructions) and had no register to spare.
//   * On 1 or 2 CTAs the member-level scan step is a branch-free, fully unrolled, predicated sum of the published
//     warp totals (two dependent-add chains) instead of a loop of dependent shared-memory loads.
//   * The cluster size is a template parameter: any size 1..8 and 16 (the non-portable maximum: 16 x 2048 points
//     hold the paper's production grid of 2^15 points).
//   * The member-level scan step leaves the critical path: the exponents of a thread's points are formed WITHOUT
//     the sum B of everything above the thread, the differences to the reference point do not contain it, and B
//     enters only the one full exponential per thread, e^{x_ref + (h/2) B}.  B itself is summed by the lanes of a
//     warp in parallel (one published total per lane, five shuffle steps) while the relative polynomials run.
//
// Per RK stage (equations PAPER.md:43-53 eqs (2)-(6); boundary conditions PAPER.md:59-75):
//   phase 1  (after sync S: neighbours' Phi, Pi edges + warp totals of f)  delta, E = e^{-delta},
//            fluxes G, H, F, eq (4) for A with its RK combine, publish H, F edges            -> sync F
//   phase 2  Kreiss-Oliger Q Phi, Q Pi and interior D4 (before the wait), edge D4, RK combine for
//            Phi, Pi, collapse test (stage 4), f of the NEW state, thread/warp scan,
//            publish Phi, Pi edges + warp totals                                             -> sync S
#pragma once
#include "adsc_internal.cuh"
#include "adsc_resident.cuh"
#include "adsc_exp.cuh"
#include "adsc_ptx.cuh"

namespace adsc {

// FIXED: the paper's second workload (Table II), A = 1 and delta = 0 held fixed: no f', no scan,
// no exponential, eq (4) not evolved, no collapse test -- the same stencils, exchanges and RK combine.
// NS: Runge-Kutta stages per step: 4 (classical RK4), 3 (Heun's third-order rule) or 2 (explicit midpoint): the
// weights come in ResConsts (R12, R25); only the stage count and the barrier phase bookkeeping differ.
template <int P, int THREADS, bool ACC_REG, int CL, bool FIXED, int NS>
__global__ void __launch_bounds__(THREADS, (THREADS * P <= 1024) ? 2 : 1) k_resident3(const __grid_constant__ ResParams prm)
{
    using L = Res3Layout<P, THREADS, ACC_REG, CL>;
    constexpr bool MULTI = CL > 1;
    constexpr int LD = L::LD, NW = L::NW, NG = L::NG, SEG = L::SEG, RX = L::RX;
    constexpr unsigned FULL = 0xffffffffu;
#ifndef ADSC_R3_EARLY
#define ADSC_R3_EARLY 0
#endif
#ifndef ADSC_R3_NFILL
#define ADSC_R3_NFILL 3
#endif
    // Scope of the acquire in the mbarrier waits that guard data written by peer CTAs: cluster (the formally required
    // one; ptxas adds an L1 invalidate, CCTL.IVALL, behind such a wait).  Measured with CTA scope instead (the data
    // lives in shared memory, which no cache holds): no difference (cfg2 0.621 -> 0.623), so the formal scope stays.
#ifndef ADSC_R3_LANESUM_MIN_NG
#define ADSC_R3_LANESUM_MIN_NG 32
#endif
    constexpr bool LANESUM = NG >= ADSC_R3_LANESUM_MIN_NG;              // member-level sum by the lanes of the warp
    constexpr bool EARLY = ADSC_R3_EARLY && (P >= 6);                   // interior right-hand sides before the sync-F wait
    constexpr int NFILL = (P < ADSC_R3_NFILL) ? P : ADSC_R3_NFILL;      // Kreiss-Oliger points computed inside the shuffle chain
    extern __shared__ __align__(16) double smem[];
    double *xPhi = smem + L::o_xPhi, *xPi = smem + L::o_xPi, *xH = smem + L::o_xH, *xF = smem + L::o_xF;
    double *tSC = smem + L::o_tSC, *tT = smem + L::o_tT, *tC = smem + L::o_tC;
    double *un = smem + L::o_un, *accS = smem + L::o_acc;
    double2 *wt = reinterpret_cast<double2 *>(smem + L::o_wt);

    const int rank = MULTI ? (int)cluster_rank() : 0;
    const int b = blockIdx.x / CL;
    MemberRec *rec = prm.rec + b;
    if (rec->collapsed || prm.nsteps <= 0) return;      // uniform over the cluster

    const Problem &pb = prm.pb;
    const ResConsts &K = prm.k;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, col = tid + 1;
    const int g0 = rank * SEG + tid * P;                 // first owned grid index
    const bool lo_edge = (tid == 0), hi_edge = (tid == THREADS - 1);
    const bool first = lo_edge && rank == 0;             // owns i = 0
    const bool last = hi_edge && rank == CL - 1;         // owns i = N-2; i = N-1 is its halo
    const int gw = rank * NW + warp;                     // my warp among the member's NG warps
    const size_t row = (size_t)b * pb.NP;

    // sync points: S is double-buffered by the parity of its index, F is single
    const uint32_t mbS0 = smem_u32(smem + L::o_mbar), mbS1 = mbS0 + 8, mbF = mbS0 + 16;
    // transaction bytes this CTA receives from its peers per sync
    const uint32_t txS = MULTI ? (uint32_t)((rank > 0 ? 48 : 0) + (rank < CL - 1 ? 48 : 0) + (FIXED ? 0 : (CL - 1) * NW * 16)) : 0u;
    const uint32_t txF = MULTI ? (uint32_t)((rank > 0 ? 32 : 0) + (rank < CL - 1 ? 32 : 0)) : 0u;
    if (tid == 0) {
        mbar_init(mbS0, NW); mbar_init(mbS1, NW); mbar_init(mbF, NW);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

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
            tC[p * THREADS + tid] = prm.tb.C[g0 + p] * K.d4c;
            if constexpr (ACC_REG) { accP[p] = ph[p]; accQ[p] = pi[p]; accA[p] = a[p]; }
            else { accS[(0 * P + p) * THREADS + tid] = ph[p]; accS[(1 * P + p) * THREADS + tid] = pi[p]; accS[(2 * P + p) * THREADS + tid] = a[p]; }
        }
        if (lo_edge) tSC[(P - 1) * LD + 0] = -2.0 * prm.tb.sc[g0 - 1];            // odd ghost at x=0
        if (hi_edge) tSC[0 * LD + THREADS + 1] = -2.0 * prm.tb.sc[g0 + P];        // 0 at x=pi/2
    }
    // mbarrier initialisation must be visible to every thread (and peer CTA) that arrives or stores on it
    if (MULTI) {
        asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    } else {
        __syncthreads();
    }

    // Kept across sync S: f' = -2 f of the own points (fo), thread-local suffix sums s_p (so), the
    // exclusive warp-level suffix (excl), and the own-point part of the Kreiss-Oliger sums (kP, kQ).
    double fo[P], so[P], excl, kP[P], kQ[P];
    int bad = 0;

    // One elected lane per warp arrives; __syncwarp orders the other lanes' shared-memory stores before it.
    auto warp_arrive = [&](uint32_t mb, uint32_t tx) {
        __syncwarp();
        if (lane == 0) {
            if (MULTI && warp == 0) mbar_arrive_expect_tx(mb, tx);
            else mbar_arrive(mb);
        }
    };

    // Own-point part of Q Phi, Q Pi (R6) of the state in ph, pi at point p; the halo part is added after sync S.
    auto ko_pt = [&](const int p) {
        double sP = K.kw[0] * ph[p], sQ = K.kw[0] * pi[p];
#pragma unroll
        for (int j = 1; j <= 3; ++j) {
            if (p - j >= 0) { sP = fma(K.kw[j], ph[p - j], sP); sQ = fma(K.kw[j], pi[p - j], sQ); }
            if (p + j < P)  { sP = fma(K.kw[j], ph[p + j], sP); sQ = fma(K.kw[j], pi[p + j], sQ); }
        }
        kP[p] = sP; kQ[p] = sQ;
    };
    // f', s of the new state; publish the state edges and the warp total for sync S with index parity jb.
    auto publish_S = [&](const int jb, const bool with_flag) {
        const uint32_t mb = jb ? mbS1 : mbS0;
        if constexpr (!FIXED) {
#pragma unroll
            for (int p = 0; p < P; ++p) fo[p] = tSC[p * LD + col] * fma(ph[p], ph[p], pi[p] * pi[p]);
            // top term of the telescoped rule: S_{N-1} = S_N = f_{N-2}/12 (f_N = -f_{N-2}, f_{N-1} = 0)
            so[P - 1] = fo[P - 1] + (last ? fo[P - 1] * (1.0 / 12.0) : 0.0);
#pragma unroll
            for (int p = P - 2; p >= 0; --p) so[p] = so[p + 1] + fo[p];
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            xPhi[k * LD + col] = ph[k]; xPi[k * LD + col] = pi[k];
            xPhi[(RX - 3 + k) * LD + col] = ph[P - 3 + k]; xPi[(RX - 3 + k) * LD + col] = pi[P - 3 + k];
        }
        if (lo_edge) {
            if (rank == 0) {            // x=0: Phi odd, Pi even (R2)
#pragma unroll
                for (int k = 1; k <= 3; ++k) { xPhi[(RX - k) * LD] = -ph[k]; xPi[(RX - k) * LD] = pi[k]; }
            } else if (MULTI) {         // right halo column of the CTA below
                const uint32_t rmb = map_rank(mb, rank - 1);
                const uint32_t rP = map_rank(smem_u32(xPhi + THREADS + 1), rank - 1);
                const uint32_t rQ = map_rank(smem_u32(xPi + THREADS + 1), rank - 1);
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    st_async_f64(rP + k * LD * 8, ph[k], rmb); st_async_f64(rQ + k * LD * 8, pi[k], rmb);
                }
            }
        }
        if (hi_edge) {
            if (rank == CL - 1) {       // x=pi/2: Phi even, Pi odd, Dirichlet values (R3, eqs 9, 10)
                xPhi[0 * LD + THREADS + 1] = 0.0;        xPi[0 * LD + THREADS + 1] = 0.0;
                xPhi[1 * LD + THREADS + 1] = ph[P - 1];  xPi[1 * LD + THREADS + 1] = -pi[P - 1];
                xPhi[2 * LD + THREADS + 1] = ph[P - 2];  xPi[2 * LD + THREADS + 1] = -pi[P - 2];
            } else if (MULTI) {         // left halo column of the CTA above
                const uint32_t rmb = map_rank(mb, rank + 1);
                const uint32_t rP = map_rank(smem_u32(xPhi), rank + 1);
                const uint32_t rQ = map_rank(smem_u32(xPi), rank + 1);
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    st_async_f64(rP + (RX - 3 + k) * LD * 8, ph[P - 3 + k], rmb);
                    st_async_f64(rQ + (RX - 3 + k) * LD * 8, pi[P - 3 + k], rmb);
                }
            }
        }
        if constexpr (FIXED) {
#pragma unroll
            for (int k = 0; k < NFILL; ++k) ko_pt(k);
        } else {
            // a2, warp level: inclusive suffix over the lanes; the warp total (and collapse flag) goes to every CTA.
            // The shuffle chain (5 dependent steps) is pure latency, so the own-point Kreiss-Oliger sums of the
            // first NFILL points are written between its steps: one basic block, ptxas interleaves them.
            double incl = so[0];
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const double o = __shfl_down_sync(FULL, incl, 1 << k);
                if (k < NFILL) ko_pt(k);
                if (lane + (1 << k) < 32) incl += o;
            }
            excl = incl - so[0];
            const double wsum = __shfl_sync(FULL, incl, 0);
            double flag = 0.0;
            if (with_flag) flag = __any_sync(FULL, bad) ? 1.0 : 0.0;
            double2 *slot = wt + jb * NG + gw;
            if (lane == 0) *slot = make_double2(wsum, flag);
            if (MULTI) {
                if (lane < CL && lane != rank)
                    st_async_f64x2(map_rank(smem_u32(slot), lane), wsum, flag, map_rank(mb, lane));
            }
        }
        warp_arrive(mb, txS);
    };
    // Own-point part of Q Phi, Q Pi (R6) for points [NFILL, P); publish_S did the first NFILL.
    auto ko_rest = [&]() {
#pragma unroll
        for (int p = NFILL; p < P; ++p) ko_pt(p);
    };

    publish_S(0, false);
    ko_rest();
    mbar_wait<MULTI>(mbS0, 0);

    long long n_done = 0;
    int collapsed = 0;
#pragma unroll 1
    for (long long n = 0; n < prm.nsteps; ++n) {
#pragma unroll 1
        for (int s = 0; s < NS; ++s) {
            // index of this stage's sync points since the kernel started; with four stages per step its low bits
            // depend on s only
            const unsigned j = (NS == 4) ? (unsigned)s : (unsigned)(n * NS + s);
            const double a_next = K.a_next[s], b_w = K.b_w[s];
            // sync S index j = 4n+s: buffer s&1; sync F index 4n+s: parity s&1
            const double2 *wts = wt + (j & 1u) * NG;

            // ---------------------------------------------------------------- phase 1 (after sync S)
            double hlP[3], hrP[3], hlQ[3], hrQ[3];    // 3 halo points per side of the stage state
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                hlP[k] = xPhi[(RX - 3 + k) * LD + col - 1]; hlQ[k] = xPi[(RX - 3 + k) * LD + col - 1];
                hrP[k] = xPhi[k * LD + col + 1];            hrQ[k] = xPi[k * LD + col + 1];
            }
            // halo part of the Kreiss-Oliger sums
#pragma unroll
            for (int p = 0; p < P; ++p) {
#pragma unroll
                for (int j = 1; j <= 3; ++j) {
                    if (p - j < 0) { kP[p] = fma(K.kw[j], hlP[3 + p - j], kP[p]); kQ[p] = fma(K.kw[j], hlQ[3 + p - j], kQ[p]); }
                    if (p + j >= P) { kP[p] = fma(K.kw[j], hrP[p + j - P], kP[p]); kQ[p] = fma(K.kw[j], hrQ[p + j - P], kQ[p]); }
                }
            }
            double E[P];
            if constexpr (FIXED) {
#pragma unroll
                for (int p = 0; p < P; ++p) E[p] = 1.0;                   // delta = 0 held fixed
            } else {
                const double scm = tSC[(P - 1) * LD + col - 1], scp = tSC[0 * LD + col + 1];
                // a2, member level: the sum B of all f' above this thread's points.  It enters only the reference
                // exponential of the thread (see exp3_near), so the sum runs beside the arithmetic below.
                double B;
                if constexpr (LANESUM) {
                    double v = 0.0;
#pragma unroll
                    for (int k = 0; k < (NG + 31) / 32; ++k) {
                        const int idx = lane + 32 * k;
                        if (idx < NG) { const double t = wts[idx].x; v += (idx > gw) ? t : 0.0; }
                    }
#pragma unroll
                    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(FULL, v, d);
                    B = excl + v;
                } else {                    // few warps: predicated serial sum (predicates are warp- / CTA-uniform)
                    double B0 = excl, B1 = 0.0;
                    const double2 *wl = wts + rank * NW;
#pragma unroll
                    for (int w = 1; w < NW; ++w) {
                        if (w > warp) { if (w & 1) B1 += wl[w].x; else B0 += wl[w].x; }
                    }
                    if (MULTI) {
#pragma unroll
                        for (int r = 1; r < CL; ++r) {
                            if (r > rank) {
#pragma unroll
                                for (int w = 0; w < NW; ++w) { if (w & 1) B1 += wts[r * NW + w].x; else B0 += wts[r * NW + w].x; }
                            }
                        }
                    }
                    B = B0 + B1;
                }
                // a1/a2: -delta_p = (h/2)(s_{p+2} + B) + (h/48)(25 f'_{p+1} + 12 f'_p - f'_{p-1}),  f' = -2 f;
                // nd holds it without the (h/2) B term
                double nd[P];
                {
                    const double fm = scm * fma(hlP[2], hlP[2], hlQ[2] * hlQ[2]);     // f'_{-1}
                    const double fp = scp * fma(hrP[0], hrP[0], hrQ[0] * hrQ[0]);     // f'_{P}
                    const double top = last ? fo[P - 1] * (1.0 / 12.0) : 0.0;         // as in publish_S
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const double f_lo = (p == 0) ? fm : fo[p - 1];
                        const double f_hi = (p == P - 1) ? fp : fo[p + 1];
                        const double s2 = (p + 2 < P) ? so[p + 2] : ((p + 2 == P) ? top : top - fp);
                        double loc = K.c25 * f_hi;
                        loc = fma(K.c12, fo[p], loc);
                        loc = fma(-K.c1, f_lo, loc);
                        nd[p] = fma(K.hh, s2, loc);
                    }
                }
                exp3_near<P, false, true, true>(nd, E, 1.0, nullptr, K.hh * B);
            }
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
                if constexpr (FIXED) kAv[p] = 0.0;                        // A = 1 held fixed
                else kAv[p] = (tSC[p * LD + col] * a[p]) * (G * pi[p]);   // eq (4): -2 sc A G Pi
            }
            if (first) kAv[0] = 0.0;                                      // A(0,t)=1, eq (8)
            // publish flux edges
            xH[0 * LD + col] = H[0]; xH[1 * LD + col] = H[1]; xH[2 * LD + col] = H[P - 2]; xH[3 * LD + col] = H[P - 1];
            xF[0 * LD + col] = F[0]; xF[1 * LD + col] = F[1]; xF[2 * LD + col] = F[P - 2]; xF[3 * LD + col] = F[P - 1];
            if (lo_edge) {
                if (rank == 0) {       // x=0: H even, F odd
                    xH[2 * LD] = H[2]; xH[3 * LD] = H[1]; xF[2 * LD] = -F[2]; xF[3 * LD] = -F[1];
                } else if (MULTI) {
                    const uint32_t rmb = map_rank(mbF, rank - 1);
                    const uint32_t rH = map_rank(smem_u32(xH + THREADS + 1), rank - 1);
                    const uint32_t rF = map_rank(smem_u32(xF + THREADS + 1), rank - 1);
                    st_async_f64(rH, H[0], rmb); st_async_f64(rH + LD * 8, H[1], rmb);
                    st_async_f64(rF, F[0], rmb); st_async_f64(rF + LD * 8, F[1], rmb);
                }
            }
            if (hi_edge) {
                if (rank == CL - 1) {  // x=pi/2: H odd with H=0 there; F even with the limit of R5
                    xH[0 * LD + THREADS + 1] = 0.0; xH[1 * LD + THREADS + 1] = -H[P - 1];
                    xF[0 * LD + THREADS + 1] = (16.0 * Gl1 - Gl2) * K.inv12h2;
                    xF[1 * LD + THREADS + 1] = F[P - 1];
                } else if (MULTI) {
                    const uint32_t rmb = map_rank(mbF, rank + 1);
                    const uint32_t rH = map_rank(smem_u32(xH), rank + 1);
                    const uint32_t rF = map_rank(smem_u32(xF), rank + 1);
                    st_async_f64(rH + 2 * LD * 8, H[P - 2], rmb); st_async_f64(rH + 3 * LD * 8, H[P - 1], rmb);
                    st_async_f64(rF + 2 * LD * 8, F[P - 2], rmb); st_async_f64(rF + 3 * LD * 8, F[P - 1], rmb);
                }
            }
            warp_arrive(mbF, txF);                                        // sync F: arrive

            // ---------------------------------------------------------------- between arrive and wait
            // a4/a5 for A (eq 4 needs no neighbour).  Invariant at the start of every step: acc == u^n == state.
            if constexpr (FIXED) {
                // A is not evolved
            } else if (s < NS - 1) {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int ui = (2 * P + p) * THREADS + tid;
                    if constexpr (ACC_REG) accA[p] = fma(b_w, kAv[p], accA[p]);
                    else accS[ui] = fma(b_w, kAv[p], accS[ui]);
                    a[p] = fma(a_next, kAv[p], un[ui]);
                }
            } else {
                bad = 0;
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int ui = (2 * P + p) * THREADS + tid;
                    double accn;
                    if constexpr (ACC_REG) { accn = fma(b_w, kAv[p], accA[p]); accA[p] = accn; }
                    else { accn = fma(b_w, kAv[p], accS[ui]); accS[ui] = accn; }
                    a[p] = accn; un[ui] = accn;
                    if (!(accn >= K.thr)) bad = 1;
                }
            }
            // interior points p in [2, P-2) need own fluxes only: their differences, right-hand sides and
            // RK combine are done before the wait, in the shadow of the slowest warp's arrival
            double dH[P], dF[P], kPs[P], kQs[P];
            // a4 + a5 for points [p0, p1): new stage state (s < 3; the accumulator update is deferred past
            // the scan) or the new time level (s = 3)
            auto rhs_combine = [&](const int p0, const int p1) {
#pragma unroll
                for (int p = p0; p < p1; ++p) {
                    const double qq = kQ[p];
                    kP[p] = fma(K.d4c, dH[p], kP[p]);
                    kQ[p] = fma(tC[p * THREADS + tid], dF[p], qq);
                    if (p == 0 && first) {       // Phi(0,t)=0 (eq 7); Pi_dot(0) = 3 (A e^{-delta} Phi)'(0) (R4)
                        kP[0] = 0.0;
                        kQ[0] = fma(8.0 * G1 - G2, K.c_org, qq);
                    }
                }
                if (s < NS - 1) {
#pragma unroll
                    for (int p = p0; p < p1; ++p) {
                        const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                        kPs[p] = kP[p]; kQs[p] = kQ[p];
                        ph[p] = fma(a_next, kP[p], un[uP]); pi[p] = fma(a_next, kQ[p], un[uQ]);
                    }
                } else {
#pragma unroll
                    for (int p = p0; p < p1; ++p) {
                        const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                        double nP, nQ;
                        if constexpr (ACC_REG) { nP = fma(b_w, kP[p], accP[p]); nQ = fma(b_w, kQ[p], accQ[p]); accP[p] = nP; accQ[p] = nQ; }
                        else { nP = fma(b_w, kP[p], accS[uP]); nQ = fma(b_w, kQ[p], accS[uQ]); accS[uP] = nP; accS[uQ] = nQ; }
                        ph[p] = nP; pi[p] = nQ; un[uP] = nP; un[uQ] = nQ;
                    }
                }
            };
#pragma unroll
            for (int p = 2; p < P - 2; ++p) {
                dH[p] = fma(8.0, H[p + 1] - H[p - 1], H[p - 2] - H[p + 2]);
                dF[p] = fma(8.0, F[p + 1] - F[p - 1], F[p - 2] - F[p + 2]);
            }
            // edge operands are taken before the interior state is overwritten (ph, pi are not flux inputs
            // any more at this point: H, F, G1, G2 hold everything phase 2 needs)
            if (EARLY) rhs_combine(2, P - 2);
            mbar_wait<MULTI>(mbF, (uint32_t)(j & 1u));                    // sync F: wait

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
            if (EARLY) { rhs_combine(0, 2); rhs_combine(P - 2, P); }
            else rhs_combine(0, P);
            const int jb = (int)((j + 1u) & 1u);                          // buffer of the next sync S
            publish_S(jb, s == NS - 1);                                   // sync S: arrive
            if (s < NS - 1) {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                    if constexpr (ACC_REG) { accP[p] = fma(b_w, kPs[p], accP[p]); accQ[p] = fma(b_w, kQs[p], accQ[p]); }
                    else { accS[uP] = fma(b_w, kPs[p], accS[uP]); accS[uQ] = fma(b_w, kQs[p], accS[uQ]); }
                }
            }
            ko_rest();                                                    // for the next stage
            mbar_wait<MULTI>(jb ? mbS1 : mbS0, (uint32_t)(((j + 1u) >> 1) & 1u));   // sync S: wait
            if (s == NS - 1) {
                // a6: collapse test of PAPER.md:85 on A^{n+1}: every warp of the member published its flag
                int any = 0;
                if constexpr (!FIXED) {
                    const int2 *fl = reinterpret_cast<const int2 *>(wt + jb * NG);
#pragma unroll
                    for (int k = 0; k < (NG + 31) / 32; ++k) {
                        const int idx = lane + 32 * k;
                        if (idx < NG) any |= fl[2 * idx + 1].y;           // high word of the flag (0.0 or 1.0)
                    }
                    any = __any_sync(FULL, any != 0);
                }
                n_done = n + 1;
                if (any && (prm.check_last || n + 1 < prm.nsteps)) collapsed = 1;
            }
        }
        if (collapsed) break;                                             // uniform over the cluster
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
    // no CTA may exit while a peer can still store into its shared memory
    if (MULTI) asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

}  // namespace adsc
