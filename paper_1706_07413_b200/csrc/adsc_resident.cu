// adsc_resident.cu — the resident RK4 kernel: one ensemble member per CTA (or per
// thread-block cluster of CL CTAs), state on chip across all four RK stages and across
// many time steps; HBM is touched once at launch and once at exit.
//
// Per RK stage (equations PAPER.md:43-53 eqs (2)-(6), boundary
// conditions PAPER.md:59-75 eqs (7)-(12)):
//   A  a1 source f and quadrature increments I, KO dissipation of Phi, Pi; a2 the delta
//      suffix scan: thread-serial over P points, warp shuffle, then ONE barrier through
//      which every warp of every CTA of the cluster publishes its total (DSMEM);
//   B  a3 fluxes G,H,F (one exp per point), a4/a5 for A (eq 4 has no stencil);
//   C  a4 centred 4th-order differences of H and F, a5 RK4 combine for Phi, Pi,
//      a6 collapse test at stage 4 folded into the stage's last barrier.
// Thread t of a CTA owns P contiguous points; only the 3 (Phi,Pi) / 2 (H,F) edge values
// go through shared memory, laid out [row p][thread] so accesses are bank-conflict free.
// Physical boundaries are closed by writing parity-mirrored values into the halo columns
// (R2-R5); inside a cluster the halo columns are written by the neighbour CTA.
#include <cooperative_groups.h>

#include "adsc_internal.cuh"
#include "adsc_resident.cuh"

namespace cg = cooperative_groups;

namespace adsc {

template <int P, int THREADS, bool ACC_REG>
struct ResLayout {
    static constexpr int SEG = P * THREADS;
    static constexpr int LD = THREADS + 2;          // halo column on each side
    static constexpr int NW = THREADS / 32;
    static constexpr int o_xPhi = 0;
    static constexpr int o_xPi = o_xPhi + P * LD;
    static constexpr int o_xH = o_xPi + P * LD;
    static constexpr int o_xF = o_xH + 4 * LD;
    static constexpr int o_tSC = o_xF + 4 * LD;
    static constexpr int o_tT = o_tSC + P * LD;
    static constexpr int o_tC = o_tT + P * THREADS;
    static constexpr int o_un = o_tC + P * THREADS;
    static constexpr int o_acc = o_un + 3 * P * THREADS;
    static constexpr int o_wtot = o_acc + (ACC_REG ? 0 : 3 * P * THREADS);
    static constexpr int o_flag = o_wtot + 2 * 64;
    static constexpr int n_doubles = o_flag + 2;
    static constexpr size_t bytes = (size_t)n_doubles * sizeof(double);
};

template <int P, int THREADS, bool ACC_REG, bool MULTI>
__global__ void __launch_bounds__(THREADS, 1) k_resident(const ResParams prm)
{
    using L = ResLayout<P, THREADS, ACC_REG>;
    constexpr int LD = L::LD, NW = L::NW, SEG = L::SEG;
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
    const size_t row = (size_t)b * pb.NP;

    // neighbour CTAs' exchange buffers (DSMEM)
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
            tSC[p * LD + col] = prm.tb.sc[g0 + p];
            tT[p * THREADS + tid] = prm.tb.T[g0 + p];
            tC[p * THREADS + tid] = prm.tb.C[g0 + p];
            if constexpr (ACC_REG) { accP[p] = 0.0; accQ[p] = 0.0; accA[p] = 0.0; }
        }
        if (lo_edge) tSC[(P - 1) * LD + 0] = prm.tb.sc[g0 - 1];
        if (hi_edge) { tSC[0 * LD + THREADS + 1] = prm.tb.sc[g0 + P]; tSC[1 * LD + THREADS + 1] = prm.tb.sc[g0 + P + 1]; }
        if (tid < 2) iflag[tid] = 0;
    }

    const double c13 = 13.0 * pb.h / 24.0, c1 = pb.h / 24.0;
    const double d4c = 1.0 / (12.0 * pb.h), koc = pb.ko_eps / (64.0 * pb.h);
    const double thr = pb.thr;

    // Publish the edge values of the stage state for the neighbours' stencils.
    auto publish_state = [&]() {
#pragma unroll
        for (int p = 0; p < P; ++p)
            if (p < 3 || p >= P - 3) { xPhi[p * LD + col] = ph[p]; xPi[p * LD + col] = pi[p]; }
        if (lo_edge) {
            if (rank == 0) {            // x=0: Phi odd, Pi even (R2)
#pragma unroll
                for (int k = 1; k <= 3; ++k) { xPhi[(P - k) * LD] = -ph[k]; xPi[(P - k) * LD] = pi[k]; }
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
                for (int k = 0; k < 3; ++k) { nb_hi_xPhi[(P - 3 + k) * LD] = ph[P - 3 + k]; nb_hi_xPi[(P - 3 + k) * LD] = pi[P - 3 + k]; }
            }
        }
    };
    auto barrier = [&]() { if (MULTI) cluster.sync(); else __syncthreads(); };

    publish_state();
    barrier();

    long long n_done = 0;
    int collapsed = 0;
    int stage_ctr = 0;
#pragma unroll 1
    for (long long n = 0; n < prm.nsteps; ++n) {
        int bad = 0;
#pragma unroll 1
        for (int s = 0; s < 4; ++s, ++stage_ctr) {
            const double a_next = (s == 2) ? pb.dt : 0.5 * pb.dt;
            const double b_w = (s == 0 || s == 3) ? pb.dt / 6.0 : pb.dt / 3.0;

            // ------------------------------------------------------------------ A
            double qP[P], qQ[P], dl[P];
            double base;
            {
                double phx[P + 6], pix[P + 6];
#pragma unroll
                for (int p = 0; p < P; ++p) { phx[p + 3] = ph[p]; pix[p + 3] = pi[p]; }
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    phx[k] = xPhi[(P - 3 + k) * LD + col - 1]; pix[k] = xPi[(P - 3 + k) * LD + col - 1];
                    phx[P + 3 + k] = xPhi[k * LD + col + 1];   pix[P + 3 + k] = xPi[k * LD + col + 1];
                }
                double f[P + 3];
#pragma unroll
                for (int k = 0; k < P + 3; ++k) {
                    double scv;
                    if (k == 0) scv = tSC[(P - 1) * LD + col - 1];
                    else if (k <= P) scv = tSC[(k - 1) * LD + col];
                    else scv = tSC[(k - P - 1) * LD + col + 1];
                    f[k] = scv * (phx[k + 2] * phx[k + 2] + pix[k + 2] * pix[k + 2]);
                }
#pragma unroll
                for (int p = P - 1; p >= 0; --p) {
                    const double I = c13 * (f[p + 1] + f[p + 2]) - c1 * (f[p] + f[p + 3]);
                    dl[p] = (p == P - 1) ? I : dl[p + 1] + I;
                }
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    qP[p] = koc * (phx[p] - 6.0 * phx[p + 1] + 15.0 * phx[p + 2] - 20.0 * phx[p + 3]
                                   + 15.0 * phx[p + 4] - 6.0 * phx[p + 5] + phx[p + 6]);
                    qQ[p] = koc * (pix[p] - 6.0 * pix[p + 1] + 15.0 * pix[p + 2] - 20.0 * pix[p + 3]
                                   + 15.0 * pix[p + 4] - 6.0 * pix[p + 5] + pix[p + 6]);
                }
                // scan: warp level, then all warps of all CTAs through one barrier
                const double incl = warp_suffix_incl(dl[0]);
                const double wsum = __shfl_sync(0xffffffffu, incl, 0);
                const int buf = (stage_ctr & 1) * 64;
                if (MULTI) {
                    if (lane < CL) cluster.map_shared_rank(wtot, lane)[buf + rank * NW + warp] = wsum;
                } else {
                    if (lane == 0) wtot[buf + warp] = wsum;
                }
                barrier();
                const int nG = NW * CL;
                double v0 = (lane < nG) ? wtot[buf + lane] : 0.0;
                double s0 = warp_suffix_incl(v0);
                double s1 = 0.0;
                if (nG > 32) {
                    double v1 = (lane + 32 < nG) ? wtot[buf + 32 + lane] : 0.0;
                    s1 = warp_suffix_incl(v1);
                    s0 += __shfl_sync(0xffffffffu, s1, 0);
                }
                const int want = rank * NW + warp + 1;          // first warp above mine
                double c0 = __shfl_sync(0xffffffffu, s0, want & 31);
                double c1v = __shfl_sync(0xffffffffu, s1, want & 31);
                const double carry = (want >= nG) ? 0.0 : (want < 32 ? c0 : c1v);
                base = (incl - dl[0]) + carry;
            }

            // ------------------------------------------------------------------ B
            double H[P], F[P], G1 = 0.0, G2 = 0.0, Gl1 = 0.0, Gl2 = 0.0;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const double delta = dl[p] + base;
                const double AE = a[p] * exp(-delta);
                const double G = AE * ph[p];
                H[p] = AE * pi[p];
                F[p] = tT[p * THREADS + tid] * G;
                if (p == 1) G1 = G;
                if (p == 2) G2 = G;
                if (p == P - 1) Gl1 = G;
                if (p == P - 2) Gl2 = G;
                double kA = -2.0 * tSC[p * LD + col] * a[p] * G * pi[p];
                if (p == 0 && first) kA = 0.0;                   // A(0,t)=1, eq (8)
                // RK4 combine for A (eq 4 needs no neighbour)
                const int ui = (2 * P + p) * THREADS + tid;
                const double bs = (s == 0) ? a[p] : un[ui];
                double accv;
                if constexpr (ACC_REG) accv = (s == 0) ? bs : accA[p];
                else accv = (s == 0) ? bs : accS[ui];
                const double accn = fma(b_w, kA, accv);
                if (s < 3) {
                    if constexpr (ACC_REG) accA[p] = accn; else accS[ui] = accn;
                    a[p] = fma(a_next, kA, bs);
                } else {
                    a[p] = accn; un[ui] = accn;
                    if (!(accn >= thr)) bad = 1;
                }
            }
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
                    xF[0 * LD + THREADS + 1] = (16.0 * Gl1 - Gl2) / (12.0 * pb.h * pb.h);
                    xF[1 * LD + THREADS + 1] = F[P - 1];
                } else if (MULTI) {
                    nb_hi_xH[2 * LD] = H[P - 2]; nb_hi_xH[3 * LD] = H[P - 1];
                    nb_hi_xF[2 * LD] = F[P - 2]; nb_hi_xF[3 * LD] = F[P - 1];
                }
            }
            barrier();

            // ------------------------------------------------------------------ C
            {
                double Hx[P + 4], Fx[P + 4];
                Hx[0] = xH[2 * LD + col - 1]; Hx[1] = xH[3 * LD + col - 1];
                Fx[0] = xF[2 * LD + col - 1]; Fx[1] = xF[3 * LD + col - 1];
                Hx[P + 2] = xH[0 * LD + col + 1]; Hx[P + 3] = xH[1 * LD + col + 1];
                Fx[P + 2] = xF[0 * LD + col + 1]; Fx[P + 3] = xF[1 * LD + col + 1];
#pragma unroll
                for (int p = 0; p < P; ++p) { Hx[p + 2] = H[p]; Fx[p + 2] = F[p]; }
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    double kP = fma(d4c, fma(8.0, Hx[p + 3] - Hx[p + 1], Hx[p] - Hx[p + 4]), qP[p]);
                    double kQ = fma(tC[p * THREADS + tid] * d4c, fma(8.0, Fx[p + 3] - Fx[p + 1], Fx[p] - Fx[p + 4]), qQ[p]);
                    if (p == 0 && first) {           // Phi(0,t)=0 (eq 7); Pi_dot(0) = 3 (A e^{-delta} Phi)'(0) (R4)
                        kP = 0.0;
                        kQ = (8.0 * G1 - G2) / (2.0 * pb.h) + qQ[0];
                    }
                    const int uP = (0 * P + p) * THREADS + tid, uQ = (1 * P + p) * THREADS + tid;
                    const double bP = (s == 0) ? ph[p] : un[uP];
                    const double bQ = (s == 0) ? pi[p] : un[uQ];
                    double aP, aQ;
                    if constexpr (ACC_REG) { aP = (s == 0) ? bP : accP[p]; aQ = (s == 0) ? bQ : accQ[p]; }
                    else { aP = (s == 0) ? bP : accS[uP]; aQ = (s == 0) ? bQ : accS[uQ]; }
                    const double nP = fma(b_w, kP, aP), nQ = fma(b_w, kQ, aQ);
                    if (s < 3) {
                        if constexpr (ACC_REG) { accP[p] = nP; accQ[p] = nQ; } else { accS[uP] = nP; accS[uQ] = nQ; }
                        ph[p] = fma(a_next, kP, bP); pi[p] = fma(a_next, kQ, bQ);
                    } else {
                        ph[p] = nP; pi[p] = nQ; un[uP] = nP; un[uQ] = nQ;
                    }
                }
            }
            publish_state();
            if (s < 3) {
                barrier();
            } else {
                // a6: collapse test of PAPER.md:85 folded into the last barrier of the step
                int any;
                if (MULTI) {
                    const int par = (int)(n & 1);
                    const int cta_bad = __syncthreads_or(bad);
                    if (cta_bad && tid < CL) cluster.map_shared_rank(iflag, tid)[par] = 1;
                    cluster.sync();
                    any = iflag[par];
                    if (tid == 0) iflag[par ^ 1] = 0;
                } else {
                    any = __syncthreads_or(bad);
                }
                n_done = n + 1;
                if (any && (prm.check_last || n + 1 < prm.nsteps)) collapsed = 1;
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
#define ADSC_RES_CFG(P_, T_, ACC_)                                                        \
    { "P" #P_ "xT" #T_ #ACC_, P_, T_, P_ * T_, ACC_, ResLayout<P_, T_, ACC_>::bytes, true, \
      { (const void *)k_resident<P_, T_, ACC_, false>, (const void *)k_resident<P_, T_, ACC_, true>,       \
        (const void *)k_resident<P_, T_, ACC_, true>, (const void *)k_resident<P_, T_, ACC_, true> } }

static const ResConfig g_cfgs1[] = {
    ADSC_RES_CFG(8, 256, true),     // SEG 2048, accumulators in registers
    ADSC_RES_CFG(4, 512, false),    // SEG 2048
    ADSC_RES_CFG(4, 256, false),    // SEG 1024
    ADSC_RES_CFG(4, 128, false),    // SEG 512
    ADSC_RES_CFG(4, 64, false),     // SEG 256
    ADSC_RES_CFG(4, 32, false),     // SEG 128
};
constexpr int n_cfgs1 = sizeof(g_cfgs1) / sizeof(g_cfgs1[0]);

// Variant index space: generation 3 (preferred), then generation 1 (any cluster size 2..8).
static int n_cfgs() { return n_cfgs3 + n_cfgs1; }
static const ResConfig &cfg_at(int k)
{
    return k < n_cfgs3 ? g_cfgs3[k] : g_cfgs1[k - n_cfgs3];
}
static const void *fn_for(const ResConfig &g, int cl, int fixed_bg, int rk_order)
{
    if (fixed_bg && rk_order != 4) return nullptr;          // not compiled: takes a streaming path
    const void *const *fn = fixed_bg ? g.fnf : (rk_order == 3 ? g.fn3 : rk_order == 2 ? g.fn2 : g.fn);
    if (cl == 1) return fn[0];
    if (g.any_cl) return fn[1];
    return cl == 2 ? fn[1] : cl == 4 ? fn[2] : cl == 8 ? fn[3] : nullptr;
}

const char *resident_cfg_name(int cfg) { return (cfg >= 0 && cfg < n_cfgs()) ? cfg_at(cfg).name : "none"; }

// Pick the widest segment that tiles N-1 with at most 8 CTAs per member (portable
// cluster limit).  Returns false if no resident configuration holds N.
bool resident_select(adsc_ctx *c)
{
    const int n_act = c->pb.N - 1;
    for (int k = 0; k < n_cfgs(); ++k) {
        const ResConfig &g = cfg_at(k);
        if (n_act % g.seg) continue;
        const int cl = n_act / g.seg;
        if (cl < 1 || cl > 8) continue;
        if (!fn_for(g, cl, c->pb.fixed_bg, c->rk_order)) continue;
        if (c->dev_smem_optin > 0 && g.smem > (size_t)c->dev_smem_optin) continue;
        c->res_cfg = k; c->cluster = cl;
        return true;
    }
    return false;
}

cudaError_t launch_resident(adsc_ctx *c, long long nsteps, int check_last)
{
    const ResConfig &g = cfg_at(c->res_cfg);
    const void *fn = fn_for(g, c->cluster, c->pb.fixed_bg, c->rk_order);
    if (!fn) return cudaErrorInvalidDeviceFunction;      // adsc_step checks this combination before launching
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem);
    if (e != cudaSuccess) return e;
    ResParams prm;
    prm.pb = c->pb; prm.tb = c->tb;
    for (int v = 0; v < 3; ++v) prm.U[v] = c->ws.U[v];
    prm.rec = c->ws.rec; prm.nsteps = nsteps; prm.check_last = check_last; prm.CL = c->cluster;
    {
        const double h = c->pb.h, dt = c->pb.dt, koc = c->pb.ko_eps / (64.0 * h);
        ResConsts &k = prm.k;
        k.d4c = 1.0 / (12.0 * h);
        k.kw[0] = -20.0 * koc; k.kw[1] = 15.0 * koc; k.kw[2] = -6.0 * koc; k.kw[3] = koc;
        k.hh = 0.5 * h; k.c25 = 25.0 * h / 48.0; k.c12 = 0.25 * h; k.c1 = h / 48.0;
        k.inv12h2 = 1.0 / (12.0 * h * h); k.c_org = 1.0 / (2.0 * h);
        rk_tableau(c->rk_order, dt, k.a_next, k.b_w);
        k.thr = c->pb.thr;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(c->pb.B * c->cluster), 1, 1);
    cfg.blockDim = dim3((unsigned)g.threads, 1, 1);
    cfg.dynamicSmemBytes = g.smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)c->cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    void *args[] = { (void *)&prm };
    e = cudaLaunchKernelExC(&cfg, fn, args);
    c->launches++;
    return e;
}

}  // namespace adsc
