// adsc_probe.cu — probes and self-tests that need no handle.  (1) adsc_selftest_exp runs the hot path's
// exponential (adsc_exp.cuh) on caller-chosen arguments and reports which of its branches ran.  (2) The two roofline denominators of the resident regime, MEASURED on the device the library runs
// on: the FP64 FMA issue rate and the shared-memory bandwidth.  bench.py runs both for
// a few tens of milliseconds before its timed region and reports them beside the derived peaks.  Nothing of the
// method's arithmetic is here.
#include "adsc_internal.cuh"
#include "adsc_exp.cuh"

namespace adsc {

// Self-test of the hot path's exponential (adsc_exp.cuh): one thread per group of 8 arguments.
__global__ void k_selftest_exp(int ngroups, const double *__restrict__ x, double *__restrict__ E, int *__restrict__ tier)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    double xv[8], Ev[8];
#pragma unroll
    for (int p = 0; p < 8; ++p) xv[p] = x[8 * g + p];
    int t = -1;
    exp3_near<8>(xv, Ev, 1.0, &t);
#pragma unroll
    for (int p = 0; p < 8; ++p) E[8 * g + p] = Ev[p];
    tier[g] = t;
}

__device__ double g_probe_sink[2];

// 16 independent FMA chains per thread (the FP64 pipe's dependent-issue latency is hidden twice over with 8 warps
// per scheduler), 2 flop per lane per instruction.
__global__ void __launch_bounds__(1024, 1) k_probe_dfma(int iters, double seed)
{
    double x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = seed + (double)(threadIdx.x + k);
    const double a = 1.0 + 1e-9 * seed, b = 1e-9;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = fma(x[k], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    if (s == 123.456) g_probe_sink[0] = s;               // never true: keeps the chains alive
}

// Conflict-free 128-bit shared-memory loads: every warp reads 512 contiguous bytes per instruction.
__global__ void __launch_bounds__(1024, 1) k_probe_lds(int iters)
{
    extern __shared__ __align__(16) double2 sm2[];
    const int n = 8192;                                  // 128 KB
    for (int k = threadIdx.x; k < n; k += blockDim.x) sm2[k] = make_double2((double)k, 1.0);
    __syncthreads();
    double2 acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = make_double2(0.0, 0.0);
    int o = threadIdx.x;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const double2 v = sm2[(o + k * 1024) & (n - 1)];
            acc[k].x += v.x; acc[k].y += v.y;
        }
        o = (o + 32) & (n - 1);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += acc[k].x + acc[k].y;
    if (s == 123.456) g_probe_sink[1] = s;
}

}  // namespace adsc

using namespace adsc;

extern "C" int adsc_selftest_exp(int ngroups, const double *h_x, double *h_E, int *h_tier)
{
    if (ngroups < 1 || ngroups > (1 << 24) || !h_x || !h_E || !h_tier) return ADSC_EINVAL;
    const size_t nb = (size_t)ngroups * 8 * sizeof(double), nt = (size_t)ngroups * sizeof(int);
    double *dx = nullptr, *dE = nullptr;
    int *dt = nullptr;
    int rc = ADSC_ECUDA;
    do {
        if (cudaMalloc(&dx, nb) != cudaSuccess || cudaMalloc(&dE, nb) != cudaSuccess || cudaMalloc(&dt, nt) != cudaSuccess) break;
        if (cudaMemcpy(dx, h_x, nb, cudaMemcpyHostToDevice) != cudaSuccess) break;
        k_selftest_exp<<<(ngroups + 127) / 128, 128>>>(ngroups, dx, dE, dt);
        if (cudaGetLastError() != cudaSuccess) break;
        if (cudaMemcpy(h_E, dE, nb, cudaMemcpyDeviceToHost) != cudaSuccess) break;
        if (cudaMemcpy(h_tier, dt, nt, cudaMemcpyDeviceToHost) != cudaSuccess) break;
        rc = ADSC_OK;
    } while (0);
    cudaFree(dx); cudaFree(dE); cudaFree(dt);
    if (rc != ADSC_OK) (void)cudaGetLastError();
    return rc;
}

extern "C" int adsc_probe(int kind, double target_ms, double *result)
{
    if (!result || !(target_ms > 0.0) || (kind != ADSC_PROBE_FP64_FMA && kind != ADSC_PROBE_SHARED_LOAD)) return ADSC_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return ADSC_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return ADSC_ECUDA;
    cudaStream_t st = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaStreamCreate(&st) != cudaSuccess) return ADSC_ECUDA;
    int rc = ADSC_ECUDA;
    const size_t smem = (kind == ADSC_PROBE_SHARED_LOAD) ? 8192 * sizeof(double2) : 0;
    do {
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        if (smem && cudaFuncSetAttribute(k_probe_lds, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) break;
        auto run = [&](int iters, float *ms) -> bool {
            if (cudaEventRecord(e0, st) != cudaSuccess) return false;
            if (kind == ADSC_PROBE_FP64_FMA) k_probe_dfma<<<sms, 1024, 0, st>>>(iters, 1.0);
            else k_probe_lds<<<sms, 1024, smem, st>>>(iters);
            if (cudaGetLastError() != cudaSuccess) return false;
            if (cudaEventRecord(e1, st) != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) return false;
            return cudaEventElapsedTime(ms, e0, e1) == cudaSuccess;
        };
        float ms = 0.f;
        int iters = 2000;
        if (!run(iters, &ms) || !run(iters, &ms)) break;              // warm-up, then calibration
        double scale = target_ms / (ms > 1e-3f ? (double)ms : 1e-3);
        if (scale > 1.0) { if (scale > 4000.0) scale = 4000.0; iters = (int)(iters * scale); }
        if (!run(iters, &ms)) break;
        const double work = (kind == ADSC_PROBE_FP64_FMA)
            ? (double)sms * 1024.0 * (double)iters * 8.0 * 16.0 * 2.0      // flop
            : (double)sms * 1024.0 * (double)iters * 8.0 * 16.0;           // bytes
        *result = work / ((double)ms * 1e-3);
        rc = ADSC_OK;
    } while (0);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaStreamDestroy(st);
    if (rc != ADSC_OK) (void)cudaGetLastError();
    return rc;
}
