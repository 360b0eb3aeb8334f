// adsc_resident.cu — host side of the resident path: which compiled configuration of the resident kernel
// (adsc_resident3.cuh) holds a member of N points, and its launch.  One ensemble member per CTA or per thread-block
// cluster of CL CTAs, the state on chip across all Runge-Kutta stages and steps of a launch; HBM is touched once at
// launch and once at exit.
#include "adsc_internal.cuh"
#include "adsc_resident.cuh"

namespace adsc {

static const void *fn_big(int cl, int kind)
{
    if (const void *f = res3_big_a(cl, kind)) return f;
    if (const void *f = res3_big_b(cl, kind)) return f;
    return res3_big_c(cl, kind);
}
static const void *fn_short(int seg, int cl, int kind)
{
    if (cl == 1) return res3_small(seg, kind);
    if (const void *f = res3_small_odd(seg, cl, kind)) return f;
    return res3_small_even(seg, cl, kind);
}
static const void *fn_1024(int cl, int kind) { return fn_short(1024, cl, kind); }
static const void *fn_512(int cl, int kind) { return fn_short(512, cl, kind); }
static const void *fn_256(int cl, int kind) { return fn_short(256, cl, kind); }
static const void *fn_128(int cl, int kind) { return cl == 1 ? res3_small(128, kind) : res3_small_odd(128, cl, kind); }

// widest segment first
static const ResConfig g_cfgs[] = {
    { "P8xT256", 8, 256, 2048, true, Res3Layout<8, 256, true, RES_MAX_CLUSTER>::bytes, fn_big },   // N-1 = cl x 2048, cl in 1..8, 16
    { "P8xT128", 8, 128, 1024, false, Res3Layout<8, 128, false, 8>::bytes, fn_1024 },                // cl = 1..5, 7, 8
    { "P4xT128", 4, 128, 512, false, Res3Layout<4, 128, false, 8>::bytes, fn_512 },
    { "P4xT64", 4, 64, 256, false, Res3Layout<4, 64, false, 8>::bytes, fn_256 },
    { "P4xT32", 4, 32, 128, false, Res3Layout<4, 32, false, 7>::bytes, fn_128 },
};
constexpr int n_cfgs = sizeof(g_cfgs) / sizeof(g_cfgs[0]);

static int kind_of(const adsc_ctx *c)
{
    if (c->pb.fixed_bg) return c->rk_order == 4 ? 1 : -1;      // (fixed background: RK4 only; other orders take a streaming path)
    return c->rk_order == 3 ? 2 : (c->rk_order == 2 ? 3 : 0);
}

const char *resident_cfg_name(int cfg) { return (cfg >= 0 && cfg < n_cfgs) ? g_cfgs[cfg].name : "none"; }

// Pick the widest segment that tiles N-1 with a cluster size the kernel is compiled for (1..8 CTAs per member, or
// 16, the non-portable maximum).  With ADSC_OPT_SPREAD and an ensemble that does not fill the device, the NARROWEST
// segment of at least 256 points whose clusters (at most 8 CTAs) still all fit on the device at once: more SMs per
// member, shorter steps.  Returns false if no resident configuration holds N.
bool resident_select(adsc_ctx *c)
{
    const int n_act = c->pb.N - 1;
    const int kind = kind_of(c);
    if (kind < 0) return false;
    const int sms = c->dev_sms > 0 ? c->dev_sms : c->sms_hint;
    int pick = -1, pick_cl = 0;
    for (int k = 0; k < n_cfgs; ++k) {
        const ResConfig &g = g_cfgs[k];
        if (n_act % g.seg) continue;
        const int cl = n_act / g.seg;
        if (cl < 1 || cl > RES_MAX_CLUSTER) continue;
        if (!g.fn(cl, kind)) continue;
        if (c->dev_smem_optin > 0 && g.smem > (size_t)c->dev_smem_optin) continue;
        if (pick < 0) { pick = k; pick_cl = cl; if (!c->spread) break; continue; }      // the default: widest segment
        // spread: a narrower segment, as long as every member's cluster has its own SMs
        if (g.seg >= 256 && cl <= c->spread_cap && (long long)c->pb.B * cl <= sms) { pick = k; pick_cl = cl; }
    }
    if (pick < 0) return false;
    c->res_cfg = pick; c->cluster = pick_cl;
    return true;
}

// Attributes and launch configuration of the selected kernel (shared by the launch and the check at adsc_bind).
static cudaError_t resident_prepare(const adsc_ctx *c, const void **pfn, cudaLaunchConfig_t *cfg, cudaLaunchAttribute *at)
{
    const ResConfig &g = g_cfgs[c->res_cfg];
    const void *fn = g.fn(c->cluster, kind_of(c));
    if (!fn) return cudaErrorInvalidDeviceFunction;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem);
    if (e != cudaSuccess) return e;
    if (c->cluster > 8) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    *cfg = cudaLaunchConfig_t{};
    cfg->gridDim = dim3((unsigned)(c->pb.B * c->cluster), 1, 1);
    cfg->blockDim = dim3((unsigned)g.threads, 1, 1);
    cfg->dynamicSmemBytes = g.smem;
    cfg->stream = c->stream;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)c->cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg->attrs = at; cfg->numAttrs = 1;
    *pfn = fn;
    return cudaSuccess;
}

// adsc_bind: can the device run at least one cluster of the selected configuration?  *clusters receives how many
// it can hold at once.
cudaError_t resident_check(adsc_ctx *c, int *clusters)
{
    const void *fn = nullptr;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    cudaError_t e = resident_prepare(c, &fn, &cfg, at);
    if (e != cudaSuccess) return e;
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, fn, &cfg);
    if (e != cudaSuccess) return e;
    *clusters = n;
    return cudaSuccess;
}

cudaError_t launch_resident(adsc_ctx *c, long long nsteps, int check_last)
{
    const void *fn = nullptr;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    cudaError_t e = resident_prepare(c, &fn, &cfg, at);
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
    void *args[] = { (void *)&prm };
    e = cudaLaunchKernelExC(&cfg, fn, args);
    c->launches++;
    return e;
}

}  // namespace adsc
