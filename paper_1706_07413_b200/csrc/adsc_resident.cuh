// adsc_resident.cuh — declarations shared by the resident kernels (adsc_resident*.cu).
#pragma once
#include "adsc_internal.cuh"

namespace adsc {

// Scalars derived from (h, dt, ko_eps, thr) on the host once per launch.  They sit in the kernel
// parameter (constant) bank, so fp64 instructions take them as c[][] operands and no register
// holds them.
struct ResConsts {
    double d4c;             // 1/(12 h)                      D4 weight
    double kw[4];           // eps_KO/(64 h) * {-20, 15, -6, 1}   KO weights by distance
    double hh;              // h/2            } telescoped delta rule for f' = -2 f
    double c25, c12, c1;    // 25h/48, h/4, h/48
    double inv12h2;         // 1/(12 h^2)     boundary flux limit (R5)
    double c_org;           // 1/(2 h)        origin l'Hopital (R4)
    double a_next[4];       // dt/2, dt/2, dt, 0      stage-state weights
    double b_w[4];          // dt/6, dt/3, dt/3, dt/6 accumulator weights
    double thr;
};

struct ResParams {
    Problem pb;
    Tables tb;
    double *U[3];
    MemberRec *rec;
    long long nsteps;
    int check_last;   // 0: the caller re-solves A after the last step and tests collapse itself
    int CL;
    ResConsts k;
};

// Shared-memory map of the resident kernel (doubles); the kernel is in adsc_resident3.cuh.
template <int P, int THREADS, bool ACC_REG, int CL>
struct Res3Layout {
    static constexpr int SEG = P * THREADS;
    static constexpr int LD = THREADS + 2;          // halo column on each side
    static constexpr int NW = THREADS / 32;
    static constexpr int NG = NW * CL;              // warps per member
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
    static constexpr int o_wt = o_acc + (ACC_REG ? 0 : 3 * P * THREADS);   // [2][NG] {total, flag}
    static constexpr int o_mbar = o_wt + 2 * NG * 2;                       // mbS[0], mbS[1], mbF, pad
    static constexpr int n_doubles = o_mbar + 4;
    static constexpr size_t bytes = (size_t)n_doubles * sizeof(double);
    static_assert(o_wt % 2 == 0, "warp-total slots must be 16-byte aligned");
};

// One compiled (points per thread, threads per CTA) configuration of the resident kernel.  fn(cl, kind) is the
// kernel for a cluster of cl CTAs per member (nullptr: not compiled); kind 0: dynamical metric, classical RK4;
// 1: fixed background A = 1, delta = 0, RK4; 2: Runge-Kutta order 3 (Heun); 3: order 2 (midpoint).
struct ResConfig {
    const char *name;
    int P, threads, seg;
    bool acc_reg;
    size_t smem;           // of the largest cluster this configuration is compiled for
    const void *(*fn)(int cl, int kind);
};
constexpr int RES_MAX_CLUSTER = 16;       // non-portable cluster size (8 is the portable limit)

// kernels are instantiated in adsc_resident3_{a,b,c,d,e}.cu
const void *res3_big_a(int cl, int kind);     // 8 points x 256 threads: clusters of 1, 2, 4
const void *res3_big_b(int cl, int kind);     // ... of 8, 16
const void *res3_big_c(int cl, int kind);     // ... of 3, 5, 6, 7
const void *res3_small(int seg, int kind);    // one CTA per member: segments of 1024, 512, 256, 128 points
const void *res3_small_odd(int seg, int cl, int kind);   // clusters of 3, 5, 7 of those segments (adsc_resident3_d.cu)
const void *res3_small_even(int seg, int cl, int kind);  // clusters of 2, 4, 8 of 1024, 512, 256 points (adsc_resident3_e.cu)

}  // namespace adsc
