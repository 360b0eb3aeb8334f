// adsc_stream_persist.cuh — declarations shared by the persistent streaming kernels
// (adsc_stream_persist.cu: 1024-point tiles, 2 or 4 points per thread; adsc_stream_persist8.cu:
// 1792-point tiles, 8 points per thread).
#pragma once
#include "adsc_internal.cuh"

namespace adsc {

constexpr int SP_CAP = 7168;                       // points per CTA chunk (3 state arrays in shared memory)
constexpr int SP_MBOX = 24;                        // doubles per chunk mailbox

struct SPConsts {
    double d4c, kw[4], hh, c25, c12, c1, inv12h2, c_org, a_next[4], b_w[4], thr;
    int ns;                          // Runge-Kutta stages: u_{s+1} = u^n + a_next[s] k_s, u^{n+1} = u^n + sum b_w[s] k_s
};

struct SPParams {
    Problem pb;
    Tables tb;
    double *U[3];
    double *ACC[3];
    MemberRec *rec;
    double *mbox;                    // [groups][2][G][SP_MBOX]
    unsigned long long *counter;     // [groups], zeroed before the launch
    long long nsteps;
    int check_last;
    int G, groups, Lc;               // chunks per member, concurrent members, points per chunk
    SPConsts k;
};

// ---- grid barrier over the G CTAs of one member (all co-resident: cooperative launch)
__device__ __forceinline__ void group_barrier(unsigned long long *cnt, unsigned long long target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(cnt, 1ULL);
        unsigned long long v;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(cnt) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

__device__ __forceinline__ double ld_cg(const double *p)
{
    double v;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}

cudaError_t launch_stream_persist8(adsc_ctx *c, const SPParams &prm);     // adsc_stream_persist8.cu

}  // namespace adsc
