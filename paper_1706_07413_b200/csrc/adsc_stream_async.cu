// adsc_stream_async.cu — persistent streaming kernel (path 1): a member too long for one cluster
// (BASELINE.json configs[3], N = 2^20+1; the paper's own grids of 2^15 and 2^16 points, PAPER.md:123,
// 169, 177) is cut into G contiguous chunks of SQ warp slices (256 points each, at most 28), one chunk
// per CTA, one CTA per SM, all co-resident (cooperative launch).
//
// What lives where:
//   shared memory   the STAGE state Phi*, Pi*, A* of the whole chunk (the three arrays every stage reads AND
//                   writes), in 16-byte chunks [tile][pair of points][thread] so that a thread's 8 contiguous
//                   points are four conflict-free 128-bit accesses and its neighbours' points are the adjacent
//                   columns; a 3-slot ring per warp that the bulk-copy engine (TMA, cp.async.bulk +
//                   mbarrier complete_tx) fills with the coefficient tables of the warp's NEXT slice
//                   while the current one is being computed
//   global (L2)     u^n and the Runge-Kutta accumulator, private to this kernel and stored PERMUTED
//                   ([slice][half][lane][4 doubles]) so that every 256-bit load/store of a warp covers
//                   1 KB of contiguous memory; the coefficient tables in the matching permuted layout
//   registers       everything of the 8 points a thread owns while their tile is in flight
//
// Per RK stage (equations PAPER.md:43-53 eqs (2)-(6); boundary conditions PAPER.md:59-75):
//   S   slice totals of f' = -2 sin x cos x (Phi^2 + Pi^2) are in shared memory -> warp 0 scans them, publishes
//       {chunk total, collapse flag, 3-point edges} to the chunk's mailbox, ONE barrier over the member's CTAs,
//       sums the totals of the chunks above (the "order dependent" integration of eq (6), is a
//       four-level suffix scan: thread / warp / slice / chunk)
//   per tile of 2048 points (8 warps x 32 lanes x 8 points), tiles in any order:
//       phase 1  delta by the telescoped rule, E = e^{-delta}, fluxes G, H, F, eq (4) with its RK combine
//                -> flux edges to the neighbour lanes (shuffles) and warps (mbarrier F, split arrive / wait)
//       phase 2  Kreiss-Oliger + D4 + RK combine for Phi, Pi, new stage state to shared memory, accumulator
//                to global memory, f' total of the NEW state for the next stage's scan
// The discrete algorithm is DESIGN.md section 1; nothing here is shared with oracle/.
#include "adsc_internal.cuh"
#include "adsc_exp.cuh"
#include "adsc_ptx.cuh"

namespace adsc {

constexpr int SA_T = 256;                 // threads per CTA
constexpr int SA_NW = SA_T / 32;          // warps
constexpr int SA_P = 8;                   // contiguous points per thread
constexpr int SA_SL = 32 * SA_P;          // points per warp slice
constexpr int SA_TILE = SA_T * SA_P;      // points per tile
constexpr int SA_MAXQ = 28;               // slices per chunk (3.5 tiles: 3 x 57 KB of state + the table ring)
constexpr int SA_RS = SA_T + 2;           // 16-byte columns per chunk row of a full tile (one halo column per side)
constexpr int SA_RS3 = SA_T / 2 + 2;      // ... of the fourth (half) tile
constexpr int SA_TS = 4 * SA_RS;          // tile stride
constexpr int SA_FS = 3 * SA_TS + 4 * SA_RS3;   // field stride (16-byte units)
// (SA_MBOX, the doubles per chunk mailbox, is in adsc_internal.cuh: the workspace layout is sized from it)
constexpr int SA_SLOT = SA_SL * 8;        // bytes of one table slice
// The two warps with the fewest slices of a ragged chunk serve the stage: SA_WS scans the slice totals, publishes the
// chunk total and computes the boundary fluxes (pre-pass); SA_WH exchanges the chunk edges and later gathers the
// totals of the other chunks.  In the top (ragged) tile, which a stage processes first, they are the idle ones.
constexpr int SA_WS = SA_NW - 1, SA_WH = SA_NW - 2;

// shared-memory map (bytes)
constexpr int SA_OFF_RING = 3 * SA_FS * 16;
constexpr int SA_OFF_MISC = SA_OFF_RING + SA_NW * 3 * SA_SLOT;
// misc region (doubles)
constexpr int o_wt = 0;                   // [32] slice totals of f'
constexpr int o_base = 32;                // [32] sum of f' over everything above the slice
constexpr int o_wfl = 64;                 // [32] slice collapse flags
constexpr int o_flo = 96;                 // [28][4] {H0, H1, F0, F1} of lane 0 of every slice
constexpr int o_fhi = o_flo + 4 * SA_MAXQ;   // [28][4] {H6, H7, F6, F7} of lane 31
constexpr int o_fpre = o_fhi + 4 * SA_MAXQ;  // [4][4] fluxes at the two points below every tile
constexpr int o_ftop = o_fpre + 16;       // [4] fluxes at the two points above the chunk
constexpr int o_xh = o_ftop + 4;          // [16] state halos of the chunk: lower Phi, Pi; upper Phi, Pi
constexpr int o_xa = o_xh + 16;           // [4] A at the two points below / above the chunk
constexpr int o_esc = o_xa + 4;           // [28][2] -2 sc just below / just above every slice
constexpr int o_etab = o_esc + 2 * SA_MAXQ;   // [5][6] tables around every boundary the pre-pass serves
constexpr int o_scal = o_etab + 32;       // [8] scalars: 0 collapse flag of the member, 1 factor C of the chunks above
constexpr int o_mbar = o_scal + 8;        // mbF, ring[8][3], mbC, mbB
constexpr int SA_MISC_DOUBLES = o_mbar + 28;
constexpr size_t SA_SMEM = (size_t)SA_OFF_MISC + (size_t)SA_MISC_DOUBLES * 8;
static_assert(SA_SMEM <= 232448, "shared memory of the streaming kernel");
static_assert(o_flo % 2 == 0 && o_fhi % 2 == 0 && o_fpre % 2 == 0 && o_ftop % 2 == 0 && o_xh % 2 == 0, "16-byte slots");

struct SAConsts {
    double d4c, kw[4], hh, c25, c12, c1, inv12h2, c_org, a_next[4], b_w[4], thr;
    int ns;                          // Runge-Kutta stages: u_{s+1} = u^n + a_next[s] k_s, u^{n+1} = u^n + sum b_w[s] k_s
};

struct SAParams {
    Problem pb;
    Tables tb;
    double *U[3];                    // [B][NP] natural layout (read at the start, written at the end of a launch)
    double *UN[3];                   // u^n, permuted
    double *ACC[3];                  // Runge-Kutta accumulator, permuted
    const double *tabp;              // [NP/256][3][256]: -2 sc, tan^2, cot^2/(12h), permuted for the ring
    MemberRec *rec;
    double *mbox;                    // [groups][2][G][SA_MBOX], zeroed before the launch (stamps start at 2)
    long long nsteps;
    int check_last;
    int G, groups, SQ;               // chunks per member, concurrent members, slices per chunk
    SAConsts k;
};

__device__ __forceinline__ double ld_cg(const double *p)
{
    double v;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}

// One 16-byte mailbox slot {value, stamp}, written and read as ONE scalar 128-bit access (PTX type .b128, relaxed, gpu
// scope; SASS STG/LDG.E.128.STRONG.GPU).  The protocol needs a reader that sees the stamp of the round to see the value
// stored with it, i.e. the 16 bytes must never tear.  A .v2.b64 access would not promise that: the PTX memory model
// treats a vector access as two separate 64-bit accesses in unspecified order.  A .b128 access is a single scalar
// operation on a naturally aligned 16-byte location; that such an access is single-copy atomic is what sm_90+ builds
// its atom.b128 on, and it is the one assumption of this protocol ("mailbox assumption").  Slots are
// 16-byte aligned by construction: the mailbox region is 256-byte aligned, SA_MBOX is even and slot offsets are even.
static_assert(SA_MBOX % 2 == 0, "mailbox slots must stay 16-byte aligned");
__device__ __forceinline__ void st_pair(double *p, double v, unsigned long long w)
{
    asm volatile("{\n\t.reg .b128 q;\n\tmov.b128 q, {%1, %2};\n\tst.relaxed.gpu.global.b128 [%0], q;\n\t}"
                 ::"l"(p), "l"(__double_as_longlong(v)), "l"(w) : "memory");
}
__device__ __forceinline__ void ld_pair(const double *p, double &v, unsigned long long &w)
{
    long long a;
    asm volatile("{\n\t.reg .b128 q;\n\tld.relaxed.gpu.global.b128 q, [%2];\n\tmov.b128 {%0, %1}, q;\n\t}"
                 : "=l"(a), "=l"(w) : "l"(p) : "memory");
    v = __longlong_as_double(a);
}

__host__ __device__ constexpr int sa_rs(int j) { return j < 3 ? SA_RS : SA_RS3; }
// 16-byte slot of point pair k (0..3) of thread t (0..255) of tile j, field f
__device__ __forceinline__ int sa_idx(int f, int j, int k, int t) { return f * SA_FS + j * SA_TS + k * sa_rs(j) + t + 1; }
// slow accessor: field f at chunk-local point l (0 <= l < chunk capacity)
__device__ __forceinline__ double sa_get(const double2 *S, int f, int l)
{
    const int j = l >> 11, r = l & (SA_TILE - 1);
    const double2 v = S[sa_idx(f, j, (r & 7) >> 1, r >> 3)];
    return (r & 1) ? v.y : v.x;
}

// Permuted layouts of one 256-point slice (point r = 8 lane + p):
//   tables, for 128-bit shared-memory reads:   double index ((p >> 1) * 32 + lane) * 2 + (p & 1)
//   u^n / accumulator, for 256-bit global accesses: double index ((p >> 2) * 32 + lane) * 4 + (p & 3)
__global__ void k_tabp(int N, int NP, Tables tb, double d4c, double *__restrict__ tabp)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= NP) return;
    const int sl = i >> 8, r = i & 255, lane = r >> 3, p = r & 7;
    const size_t o = (size_t)sl * 768 + ((p >> 1) * 32 + lane) * 2 + (p & 1);
    const bool in = i <= N - 1;
    tabp[o] = in ? -2.0 * tb.sc[i] : 0.0;
    tabp[o + 256] = (i <= N - 2) ? tb.T[i] : 0.0;
    tabp[o + 512] = (i >= 1 && i <= N - 2) ? tb.C[i] * d4c : 0.0;
}

// FIXED: A = 1, delta = 0 held fixed (Table II): no f', no scan, E = 1, eq (4) not evolved, no
// collapse test; the mailboxes then carry only the state edges.
template <bool FIXED>
__global__ void __launch_bounds__(SA_T, 1) k_stream_async(const __grid_constant__ SAParams prm)
{
    constexpr int P = SA_P;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(128) unsigned char smraw[];
    double2 *S = reinterpret_cast<double2 *>(smraw);
    double *misc = reinterpret_cast<double *>(smraw + SA_OFF_MISC);
    double *wt = misc + o_wt, *base = misc + o_base, *wfl = misc + o_wfl;
    double2 *flo2 = reinterpret_cast<double2 *>(misc + o_flo), *fhi2 = reinterpret_cast<double2 *>(misc + o_fhi);
    double2 *fpre2 = reinterpret_cast<double2 *>(misc + o_fpre), *ftop2 = reinterpret_cast<double2 *>(misc + o_ftop);
    double *xh = misc + o_xh, *xa = misc + o_xa, *esc = misc + o_esc, *etab = misc + o_etab, *scal = misc + o_scal;
    const double2 *xh2 = reinterpret_cast<const double2 *>(xh);

    const Problem &pb = prm.pb;
    const SAConsts &K = prm.k;
    const int NS = K.ns, LS = K.ns - 1;
    const int N = pb.N, G = prm.G;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int gi = blockIdx.x / G, c = blockIdx.x - gi * G;
    if (gi >= prm.groups) return;
    const int Lc = prm.SQ * SA_SL;
    const int ci0 = c * Lc;                              // first grid index of the chunk
    const int npts = min(Lc, (N - 1) - ci0);             // owned points (i = N-1 is a halo): a multiple of 8, >= 8
    const int NQ = (npts + SA_SL - 1) / SA_SL;           // slices
    const int NT = (NQ + SA_NW - 1) / SA_NW;             // tiles
    const int n_my = (NQ > warp) ? (NQ - 1 - warp) / SA_NW + 1 : 0;   // this warp owns slices 8 j + warp, j < n_my
    const bool phys_lo = (c == 0), phys_hi = (c == G - 1);
    const int cs0 = c * prm.SQ;                          // first slice of the chunk within a member row
    unsigned stage_ctr = 0;                              // barrier rounds so far; runs on across members, so the
                                                         // mailbox parity never repeats early

    const uint32_t mbF = smem_u32(misc + o_mbar);
    const uint32_t mbR = mbF + 8 + (uint32_t)warp * 24;  // this warp's three ring barriers
    const uint32_t mbC = mbF + 8 * 25;                   // "the factor of the chunks above is in shared memory"
    const uint32_t mbB = mbF + 8 * 26;                   // "slice bases and chunk halos are in shared memory"
    const uint32_t ringw = smem_u32(smraw + SA_OFF_RING) + (uint32_t)warp * 3 * SA_SLOT;
    const double2 *slot = reinterpret_cast<const double2 *>(smraw + SA_OFF_RING + (size_t)warp * 3 * SA_SLOT);
    if (tid == 0) {
        mbar_init(mbF, SA_NW);
        for (int k = 0; k < 3 * SA_NW; ++k) mbar_init(mbF + 8 + 8 * k, 1);
        mbar_init(mbC, 1);
        mbar_init(mbB, 2);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // columns of threads that own no point are read as halos by their neighbours: keep them finite
    for (int k = tid; k < 3 * SA_FS; k += SA_T) S[k] = make_double2(0.0, 0.0);
    // tables around the boundaries the pre-pass serves (chunk bottom, tile bottoms, chunk top) and at slice edges
    if (tid < 30) {
        const int m = tid / 6, k = tid - 6 * m;
        const int ib = (m < 4) ? m * SA_TILE - 3 : npts - 1;
        double v = 0.0;
        if (k < 4) { const int g = ci0 + ib + k; if (!FIXED && g >= 0 && g <= N - 1) v = -2.0 * prm.tb.sc[g]; }
        else { const int g = ci0 + ib + 1 + (k - 4); if (g >= 0 && g <= N - 2) v = prm.tb.T[g]; }
        etab[tid] = v;
    } else if (tid >= 32 && tid < 32 + 2 * NQ) {
        const int q = (tid - 32) >> 1, side = (tid - 32) & 1;
        const int g = ci0 + SA_SL * (q + side) - (side ? 0 : 1);
        esc[tid - 32] = (!FIXED && g >= -1 && g <= N - 1) ? -2.0 * prm.tb.sc[g] : 0.0;
    } else if (tid >= 128 && tid < 132) {
        misc[o_ftop + tid - 128] = 0.0;       // read (and discarded) by dead lanes of the top chunk: keep it finite
    }
    __syncthreads();

    // ---- table ring: slot t of this warp holds table t (0: -2 sc, 1: tan^2, 2: cot^2/(12h)) of the slice the warp
    // works on next; it is refilled by one bulk copy as soon as the warp has read it.  A warp with a single slice
    // keeps its tables for the whole launch.
    unsigned phs = 0;                                    // phase parities: bits 0..2 ring slots, 3 mbF, 4 mbC
    const bool reload = n_my > 1;
    auto ring_issue = [&](int t, int qn) {               // first fill: nobody has read the slot yet
        if (lane == 0)
            bulk_g2s_arrive(ringw + t * SA_SLOT, prm.tabp + ((size_t)(cs0 + qn) * 3 + t) * SA_SL, SA_SLOT, mbR + 8 * t);
    };
    if (n_my > 0) {
        const int q0 = SA_NW * (n_my - 1) + warp;
        if (!FIXED) ring_issue(0, q0);
        ring_issue(1, q0); ring_issue(2, q0);
    }
    auto ring_wait = [&](int t) { mbar_wait<false>(mbR + 8 * t, (phs >> t) & 1u); };
    // After the warp has read slot t of slice q (tile j): fetch the same table of its next slice.  The copy engine
    // (async proxy) is not ordered behind the warp's shared-memory loads (generic proxy): without an explicit order a
    // queued load could read the NEXT slice's table (seen in round 2 as a run-to-run difference).  The documented
    // order: __syncwarp (every lane's loads of the slots are done and cumulative to lane 0), then
    // fence.proxy.async.shared::cta in the issuing lane, then arrive + copy.  One warp barrier and one proxy fence per
    // slice serve all three slots: their refills are issued together once the last table (t = 2) has been read; the
    // warp's next slice starts long after that.  (Round 2 ordered each refill by predicating the copy on the arrive
    // token and making its byte count data-dependent on the loaded words -- instruction-issue order, which PTX does not
    // promise; the fenced form is also 3 % faster on cfg4, 5 % on paper32k.)
    auto ring_next = [&](int t, int j) {
        if (reload) {
            if (t == 2) {
                const int qn = SA_NW * (j > 0 ? j - 1 : n_my - 1) + warp;
                __syncwarp();
                if (lane == 0) {
                    fence_proxy_async_smem();
                    for (int u = FIXED ? 1 : 0; u < 3; ++u)
                        bulk_g2s_arrive(ringw + u * SA_SLOT, prm.tabp + ((size_t)(cs0 + qn) * 3 + u) * SA_SL, SA_SLOT, mbR + 8 * u);
                }
            }
            phs ^= 1u << t;
        }
    };

    auto warp_arrive = [&](uint32_t mbx) {
        __syncwarp();
        if (lane == 0) mbar_arrive(mbx);
    };
    // a2, chunk level.  The chunks above this one enter delta only through ONE number, the sum cs of their totals of
    // f', and e^{-delta} = C e^{-delta_local} with C = e^{(h/2) cs}: every flux of the chunk is linear in C.  So a stage
    // does not wait for the other CTAs before it starts: it works with delta_local, and one warp collects the totals
    // (stamped mailbox slots, see st_pair) when the first tile of the stage is about to need C -- by then the
    // other CTAs have long published theirs.  The warp leaves the collapse flag of the member and C in shared
    // memory and arrives on mbC.  e^0 = 1 exactly: pure AdS stays bit-exact.
    auto gather = [&](const int par) {
        const double *all = prm.mbox + ((size_t)gi * 2 + par) * G * SA_MBOX;
        double cs = 0.0;
        int fls = 0;
        for (int cc = lane; cc < G; cc += 32) {
            double t;
            unsigned long long w;
            do { ld_pair(all + (size_t)cc * SA_MBOX, t, w); } while ((w >> 1) != (unsigned long long)stage_ctr);
            if (cc > c) cs += t;
            fls |= (int)(w & 1ULL);
        }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) cs += __shfl_xor_sync(FULL, cs, d);
        fls = __any_sync(FULL, fls);
        if (lane == 0) { scal[0] = fls ? 1.0 : 0.0; scal[1] = exp3_ref(K.hh * cs); }
        warp_arrive(mbC);
    };

    for (int b = gi; b < pb.B; b += prm.groups) {
        MemberRec *rec = prm.rec + b;
        if (rec->collapsed || prm.nsteps <= 0) continue;             // uniform over the group
        const size_t row = (size_t)b * pb.NP;
        const size_t prow = row + (size_t)ci0;                       // the chunk in the permuted arrays

        // ---- load the chunk: natural layout -> shared memory (stage state) and the permuted u^n; slice totals
        for (int j = 0; j < n_my; ++j) {
            const int q = SA_NW * j + warp, l0 = q * SA_SL + lane * P;
            const int R = sa_rs(j);
            double tot = 0.0;
            double v[3][P];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double *src = prm.U[f] + row + ci0 + l0;
                ldg256(src, v[f][0], v[f][1], v[f][2], v[f][3]);
                ldg256(src + 4, v[f][4], v[f][5], v[f][6], v[f][7]);
            }
            if (l0 >= npts) {                                        // dead lanes: pure AdS, whatever the row padding holds
#pragma unroll
                for (int p = 0; p < P; ++p) { v[0][p] = 0.0; v[1][p] = 0.0; v[2][p] = 1.0; }
            }
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                double2 *d = S + sa_idx(f, j, 0, tid);
#pragma unroll
                for (int k = 0; k < 4; ++k) d[k * R] = make_double2(v[f][2 * k], v[f][2 * k + 1]);
                double *un = prm.UN[f] + prow + (size_t)q * SA_SL + lane * 4;
                stg256(un, v[f][0], v[f][1], v[f][2], v[f][3]);
                stg256(un + 128, v[f][4], v[f][5], v[f][6], v[f][7]);
            }
            if constexpr (!FIXED) {
                const double2 *tp = reinterpret_cast<const double2 *>(prm.tabp + (size_t)(cs0 + q) * 3 * SA_SL) + lane;
                double f7 = 0.0;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double2 m = tp[k * 32];
                    const double fa = m.x * fma(v[0][2 * k], v[0][2 * k], v[1][2 * k] * v[1][2 * k]);
                    const double fb = m.y * fma(v[0][2 * k + 1], v[0][2 * k + 1], v[1][2 * k + 1] * v[1][2 * k + 1]);
                    tot += fa + fb;
                    if (k == 3) f7 = fb;
                }
                if (phys_hi && l0 + P == npts) tot += f7 * (1.0 / 12.0);    // top term of the telescoped rule
                const double incl = warp_suffix_incl(tot);
                if (lane == 0) { wt[q] = incl; wfl[q] = 0.0; }
            }
        }
        int collapsed = 0;
        int n = 0;                                                   // (the host splits calls of more than 2^30 steps)

        for (;;) {
            for (int s = 0; s < NS; ++s) {
                const int par = (int)(stage_ctr & 1u);                   // mailbox buffer of this round
                ++stage_ctr;
                __syncthreads();                                         // S1: state, slice totals, flags of every tile
                if (warp == SA_WS) {
                    // ---- a2, slice level: exclusive suffix over the chunk's slices; the chunk total (with the collapse
                    // flag in the low bit of its stamp) goes to the chunk's mailbox.  Every 16-byte mailbox slot is
                    // {value, stamp of the round}: one 128-bit store / load each, no fence, no counter, no atomics.
                    double *mbx = prm.mbox + (size_t)gi * 2 * G * SA_MBOX;
                    double *mine = mbx + ((size_t)par * G + c) * SA_MBOX;
                    double exq = 0.0;
                    if constexpr (!FIXED) {
                        const double v = (lane < NQ) ? wt[lane] : 0.0;
                        const double incl = warp_suffix_incl(v);
                        exq = incl - v;
                        const double fl = (lane < NQ) ? wfl[lane] : 0.0;
                        const int anyf = __any_sync(FULL, fl != 0.0);
                        if (lane == 0) st_pair(mine, incl, 2ULL * stage_ctr + (anyf ? 1ULL : 0ULL));
                        if (lane < NQ) base[lane] = exq;                   // within the chunk (see `gather`)
                    }
                    warp_arrive(mbB);
                    asm volatile("bar.sync 1, 64;" ::: "memory");        // the chunk halos (warp SA_WH) are in shared memory
                    // ---- pre-pass: fluxes at the two points below every tile of the chunk and above the chunk, which
                    // the owner computes later in this stage or in another CTA (one lane per point, full exponential)
                    if (lane < 10) {
                        const int m = lane >> 1, e = lane & 1;
                        const bool top = (m == 4);
                        const bool valid = top ? !phys_hi : (m == 0 ? !phys_lo : m < NT);
                        if (valid) {
                            const int ib = top ? npts - 1 : m * SA_TILE - 3;
                            const int i = ib + 1 + e;
                            double fq[3], Pc = 0.0, Qc = 0.0;
    #pragma unroll
                            for (int d = 0; d < 3; ++d) {
                                const int l = ib + e + d;
                                double pv, qv;
                                if (l < 0) { pv = xh[4 + l]; qv = xh[8 + l]; }
                                else if (l >= npts) { pv = xh[8 + l - npts]; qv = xh[12 + l - npts]; }
                                else { pv = sa_get(S, 0, l); qv = sa_get(S, 1, l); }
                                fq[d] = FIXED ? 0.0 : etab[6 * m + e + d] * fma(pv, pv, qv * qv);
                                if (d == 1) { Pc = pv; Qc = qv; }
                            }
                            double Ev = 1.0, Av = 1.0;
                            if constexpr (!FIXED) {
                                double Rp2;
                                if (top) Rp2 = base[NQ - 1] - fq[1] - fq[2] - (e ? fq[0] : 0.0);
                                else { const double Rb = base[SA_NW * m] + wt[SA_NW * m]; Rp2 = e ? Rb - fq[2] : Rb; }
                                double loc = K.c25 * fq[2];
                                loc = fma(K.c12, fq[1], loc);
                                loc = fma(-K.c1, fq[0], loc);
                                Ev = exp3_ref(fma(K.hh, Rp2, loc));
                                Av = (i < 0) ? xa[2 + i] : (i >= npts ? xa[2 + i - npts] : sa_get(S, 2, i));
                            }
                            const double AE = Av * Ev, Gv = AE * Pc;
                            double *dst = top ? (misc + o_ftop) : (misc + o_fpre + 4 * m);
                            dst[e] = AE * Qc;
                            dst[2 + e] = etab[6 * m + 4 + e] * Gv;
                        }
                    }
                } else if (warp == SA_WH) {
                    // ---- state edges of the chunk to its mailbox; halo columns at the tile boundaries inside the chunk
                    // (the tile below a boundary is full); the neighbours' edges, or the parity ghosts, to shared memory
                    double *mbx = prm.mbox + (size_t)gi * 2 * G * SA_MBOX;
                    double *mine = mbx + ((size_t)par * G + c) * SA_MBOX;
                    const unsigned long long stamp = 2ULL * stage_ctr;
                    if (lane < 16 && G > 1) {
                        // slots 1..8: Phi, Pi at the first three points, A at the first two; 9..16: the same at the last
                        const int hi = lane >> 3, k = lane & 7;
                        const int f = (k < 3) ? 0 : (k < 6 ? 1 : 2), off = (k < 3) ? k : (k < 6 ? k - 3 : k - 6);
                        const int l = hi ? npts - (f == 2 ? 2 : 3) + off : off;
                        if (!(FIXED && f == 2)) st_pair(mine + 2 * (1 + lane), sa_get(S, f, l), stamp);
                    }
                    if (lane < 24) {
                        const int jb = 1 + (lane >> 3), r = lane & 7, f = r & 1, wh = r >> 1;
                        if (jb < NT) {
                            if (wh < 2) S[sa_idx(f, jb, 2 + wh, -1)] = S[sa_idx(f, jb - 1, 2 + wh, SA_T - 1)];
                            else S[sa_idx(f, jb - 1, wh - 2, SA_T)] = S[sa_idx(f, jb, wh - 2, 0)];
                        }
                    }
                    if (lane < 16) {
                        // lanes 0..7: what lies below the chunk (the LAST points of chunk c-1), 8..15: above (the FIRST of c+1)
                        const int up = lane >> 3, k = lane & 7;
                        const int f = (k < 3) ? 0 : (k < 6 ? 1 : 2), off = (k < 3) ? k : (k < 6 ? k - 3 : k - 6);
                        double v;
                        if (up ? !phys_hi : !phys_lo) {
                            const double *src = mbx + ((size_t)par * G + (up ? c + 1 : c - 1)) * SA_MBOX + 2 * (1 + (up ? 0 : 8) + k);
                            unsigned long long w = 0;
                            v = 0.0;
                            if (!(FIXED && f == 2)) { do { ld_pair(src, v, w); } while (w != stamp); }
                        } else if (!up) {                                // x = 0: Phi odd, Pi even (R2); slot off is point off-3
                            v = (f == 2) ? 1.0 : (f == 0 ? -sa_get(S, 0, 3 - off) : sa_get(S, 1, 3 - off));
                        } else {                                         // x = pi/2: Phi even, Pi odd, both zero there (R3)
                            v = (f == 2) ? 1.0 : (off == 0 ? 0.0 : (f == 0 ? sa_get(S, 0, npts - off) : -sa_get(S, 1, npts - off)));
                        }
                        if (f == 2) xa[2 * up + off] = v;
                        else xh[8 * up + 4 * f + (up ? 0 : 1) + off] = v;
                    }
                    warp_arrive(mbB);
                    asm volatile("bar.sync 1, 64;" ::: "memory");
                }
                // S2: bases (SA_WS) and halos (SA_WH) are there.  The pre-pass of SA_WS runs on beside the first tile:
                // its results are read in phase 2, behind the tile's sync F, on which SA_WS arrives after the pre-pass;
                // it reads the state of tiles that nobody changes before that sync.
                mbar_wait<false>(mbB, (uint32_t)par);    // one phase per barrier round: its parity is the mailbox parity
                if (s == 0 && n == prm.nsteps) {                         // final flag round only: nothing to overlap
                    if constexpr (!FIXED) {
                        const uint32_t cpar = (phs >> 4) & 1u;
                        phs ^= 16u;
                        if (warp == SA_WH) gather(par);
                        mbar_wait<false>(mbC, cpar);
                        // a6: collapse test of PAPER.md:85 on the state after n steps (flags of every chunk)
                        if (n > 0 && scal[0] != 0.0) collapsed = 1;
                    }
                    break;
                }

                // ---- tiles
                double Cst = 1.0;                                         // C, once this stage's gather is done
                const uint32_t cpar = (phs >> 4) & 1u;
                phs ^= 16u;
                bool tile1 = true, tile2 = false;                         // the stage's first / second tile (no reload of NT)
                for (int j = (NQ + SA_NW - 1) / SA_NW - 1; j >= 0; --j) {
                    // the first tile of the stage works with delta_local and takes C in at its end
                    const bool defer = !FIXED && tile1;
                    const bool after_defer = tile2;
                    tile2 = tile1; tile1 = false;
                    if (j >= n_my) {                                      // ragged top tile: nothing to do for this warp
                        if (defer) {
                            if (warp == SA_WH) gather(par);
                            mbar_wait<false>(mbC, cpar);
                            Cst = scal[1];
                            if (s == 0 && n > 0 && scal[0] != 0.0) { collapsed = 1; break; }     // a6
                        }
                        const uint32_t fpar = (phs >> 3) & 1u;
                        phs ^= 8u;
                        warp_arrive(mbF);
                        mbar_wait<false>(mbF, fpar);
                        continue;
                    }
                    const int q = SA_NW * j + warp;
                    const int l0 = q * SA_SL + lane * P;
                    const int tch = l0 >> 3;                              // chunk-level thread index
                    const bool live = l0 < npts;
                    const bool first = phys_lo && tch == 0;               // owns i = 0
                    const bool last = phys_hi && l0 + P == npts;          // owns i = N-2; i = N-1 is its halo
                    const int R = sa_rs(j);
                    // dead lanes (points beyond i = N-2 in the top chunk) keep their (zero) state: weights 0
                    const double a_next = live ? K.a_next[s] : 0.0, b_w = live ? K.b_w[s] : 0.0;
                    double2 *sP = S + sa_idx(0, j, 0, tid);
                    // permuted u^n / accumulator of this thread's points
                    const size_t po = prow + (size_t)q * SA_SL + lane * 4;

                    // ------------------------------------------------------------ phase 1
                    double ph[P], pi[P];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const double2 x = sP[k * R], y = sP[SA_FS + k * R];
                        ph[2 * k] = x.x; ph[2 * k + 1] = x.y; pi[2 * k] = y.x; pi[2 * k + 1] = y.y;
                    }
                    double hlP[3], hrP[3], hlQ[3], hrQ[3];                // 3 halo points per side of the stage state
                    {
                        const double2 *l2 = sP - 1 + 2 * R, *l3 = sP - 1 + 3 * R, *h0 = sP + 1, *h1 = sP + 1 + R;
                        int fol = SA_FS, foh = SA_FS;
                        if (tch == 0) { l2 = xh2; l3 = xh2 + 1; fol = 2; }
                        if (l0 + P == npts) { h0 = xh2 + 4; h1 = xh2 + 5; foh = 2; }
                        const double2 u2 = l2[0], u3 = l3[0], w2 = l2[fol], w3 = l3[fol];
                        hlP[0] = u2.y; hlP[1] = u3.x; hlP[2] = u3.y; hlQ[0] = w2.y; hlQ[1] = w3.x; hlQ[2] = w3.y;
                        const double2 v0 = h0[0], v1 = h1[0], y0 = h0[foh], y1 = h1[foh];
                        hrP[0] = v0.x; hrP[1] = v0.y; hrP[2] = v1.x; hrQ[0] = y0.x; hrQ[1] = y0.y; hrQ[2] = y1.x;
                    }
                    double m2[P], fm = 0.0, fp = 0.0;
                    if constexpr (FIXED) {
#pragma unroll
                        for (int p = 0; p < P; ++p) m2[p] = 0.0;
                    } else {
                        ring_wait(0);
#pragma unroll
                        for (int k = 0; k < 4; ++k) { const double2 m = slot[k * 32 + lane]; m2[2 * k] = m.x; m2[2 * k + 1] = m.y; }
                        const double scm = (lane == 0) ? esc[2 * q] : slot[3 * 32 + lane - 1].y;
                        const double scp = (lane == 31) ? esc[2 * q + 1] : slot[lane + 1].x;
                        ring_next(0, j);
                        fm = scm * fma(hlP[2], hlP[2], hlQ[2] * hlQ[2]);          // f'_{-1}
                        fp = scp * fma(hrP[0], hrP[0], hrQ[0] * hrQ[0]);          // f'_{P}
                    }
                    // Kreiss-Oliger sums Q Phi, Q Pi (R6): the last use of the halo points
                    double kP[P], kQ[P];
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        double sP_ = K.kw[0] * ph[p], sQ_ = K.kw[0] * pi[p];
#pragma unroll
                        for (int d = 1; d <= 3; ++d) {
                            const double pm = (p - d >= 0) ? ph[p - d] : hlP[3 + p - d], pp = (p + d < P) ? ph[p + d] : hrP[p + d - P];
                            const double qm = (p - d >= 0) ? pi[p - d] : hlQ[3 + p - d], qp = (p + d < P) ? pi[p + d] : hrQ[p + d - P];
                            sP_ = fma(K.kw[d], pm, sP_); sP_ = fma(K.kw[d], pp, sP_);
                            sQ_ = fma(K.kw[d], qm, sQ_); sQ_ = fma(K.kw[d], qp, sQ_);
                        }
                        kP[p] = sP_; kQ[p] = sQ_;
                    }
                    double E[P];
                    if constexpr (FIXED) {
#pragma unroll
                        for (int p = 0; p < P; ++p) E[p] = 1.0;                   // delta = 0 held fixed
                    } else {
                        double fo[P], so[P];
#pragma unroll
                        for (int p = 0; p < P; ++p) fo[p] = m2[p] * fma(ph[p], ph[p], pi[p] * pi[p]);
                        // top term of the telescoped rule: S_{N-1} = S_N = f_{N-2}/12 (f_N = -f_{N-2}, f_{N-1} = 0)
                        const double top = last ? fo[P - 1] * (1.0 / 12.0) : 0.0;
                        so[P - 1] = fo[P - 1] + top;
#pragma unroll
                        for (int p = P - 2; p >= 0; --p) so[p] = so[p + 1] + fo[p];
                        // a2, warp level: exclusive suffix over the lanes (the shuffle chain overlaps the arithmetic around it)
                        const double st = live ? so[0] : 0.0;             // (dead lanes may hold anything)
                        const double B = warp_suffix_incl(st) - st + base[q];
                        // a1/a2: -delta_p = (h/2)(s_{p+2} + B) + (h/48)(25 f'_{p+1} + 12 f'_p - f'_{p-1}),  f' = -2 f
                        double nd[P];
#pragma unroll
                        for (int p = 0; p < P; ++p) {
                            const double f_lo = (p == 0) ? fm : fo[p - 1];
                            const double f_hi = (p == P - 1) ? fp : fo[p + 1];
                            const double s2 = (p + 2 < P) ? so[p + 2] : ((p + 2 == P) ? top : top - fp);
                            double loc = K.c25 * f_hi;
                            loc = fma(K.c12, fo[p], loc);
                            loc = fma(-K.c1, f_lo, loc);
                            nd[p] = fma(K.hh, s2 + B, loc);
                        }
                        if (defer) exp3_near<P, false, false, true>(nd, E);
                        else exp3_near<P, true, false, true>(nd, E, Cst);
                    }
                    // global operands of the A update (needed at the end of phase 1)
                    double unA[P], acA[P];
                    if constexpr (!FIXED) {
                        if (s > 0) {
                            ldg256(prm.ACC[2] + po, acA[0], acA[1], acA[2], acA[3]);
                            ldg256(prm.ACC[2] + po + 128, acA[4], acA[5], acA[6], acA[7]);
                            if (s < LS) {
                                ldg256(prm.UN[2] + po, unA[0], unA[1], unA[2], unA[3]);
                                ldg256(prm.UN[2] + po + 128, unA[4], unA[5], unA[6], unA[7]);
                            }
                        }
                    }
                    // a3 fluxes
                    double H[P], F[P], kAv[P], a[P], Gorg = 0.0, Gtop = 0.0;   // 8 G_1 - G_2 (R4) and 16 G_{P-1} - G_{P-2} (R5)
                    {
                        ring_wait(1);
                        double tT[P];
#pragma unroll
                        for (int k = 0; k < 4; ++k) { const double2 m = slot[128 + k * 32 + lane]; tT[2 * k] = m.x; tT[2 * k + 1] = m.y; }
                        ring_next(1, j);
                        // the stage state is read again (it is still unchanged in shared memory) rather than kept in
                        // registers across the exponentials
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const double2 x = sP[k * R], y = sP[SA_FS + k * R];
                            ph[2 * k] = x.x; ph[2 * k + 1] = x.y; pi[2 * k] = y.x; pi[2 * k + 1] = y.y;
                            if constexpr (!FIXED) { const double2 z = sP[2 * SA_FS + k * R]; a[2 * k] = z.x; a[2 * k + 1] = z.y; }
                            else { a[2 * k] = 1.0; a[2 * k + 1] = 1.0; }
                        }
#pragma unroll
                        for (int p = 0; p < P; ++p) {
                            const double AE = a[p] * E[p];
                            const double Gv = AE * ph[p];
                            H[p] = AE * pi[p];
                            F[p] = tT[p] * Gv;
                            if (p == 1) Gorg = 8.0 * Gv;
                            if (p == 2) Gorg -= Gv;
                            if (p == P - 2) Gtop = -Gv;
                            if (p == P - 1) Gtop = fma(16.0, Gv, Gtop);
                            if constexpr (FIXED) kAv[p] = 0.0;                    // A = 1 held fixed
                            else kAv[p] = (m2[p] * a[p]) * (Gv * pi[p]);          // eq (4): -2 sc A G Pi
                        }
                    }
                    if (first) kAv[0] = 0.0;                                      // A(0,t)=1, eq (8)
                    if (defer) {
                        if (warp == SA_WH) gather(par);
                        mbar_wait<false>(mbC, cpar);
                        Cst = scal[1];
                        if (s == 0 && n > 0 && scal[0] != 0.0) {                  // a6: nothing has been changed yet
                            if (reload) {
                                // Slots 0 and 1 have been read and their phase bits advanced, but no refill has been
                                // issued yet (ring_next issues all three behind the read of slot 2, which is still
                                // ahead): the ring still holds this first slice's tables, which is what the next
                                // member starts with.  Take the two phase bits back.
                                if (!FIXED) phs ^= 1u;
                                phs ^= 2u;
                            }
                            collapsed = 1;
                            break;
                        }
                    }
                    const double Cl = defer ? Cst : 1.0;                          // what is still to be multiplied in
                    const double a_nC = a_next * Cl, b_wC = b_w * Cl;
                    // a4/a5 for A (eq 4 needs no neighbour)
                    if constexpr (!FIXED) {
                        double aN[P];
                        if (s < LS) {
                            double accn[P];
#pragma unroll
                            for (int p = 0; p < P; ++p) {
                                accn[p] = fma(b_wC, kAv[p], (s == 0) ? a[p] : acA[p]);
                                aN[p] = fma(a_nC, kAv[p], (s == 0) ? a[p] : unA[p]);
                            }
                            stg256(prm.ACC[2] + po, accn[0], accn[1], accn[2], accn[3]);
                            stg256(prm.ACC[2] + po + 128, accn[4], accn[5], accn[6], accn[7]);
                            if (lane == 0) wfl[q] = 0.0;
                        } else {
                            int bad = 0;
#pragma unroll
                            for (int p = 0; p < P; ++p) {
                                aN[p] = fma(b_wC, kAv[p], acA[p]);
                                if (!(aN[p] >= K.thr)) bad = 1;                   // a6
                            }
                            stg256(prm.UN[2] + po, aN[0], aN[1], aN[2], aN[3]);
                            stg256(prm.UN[2] + po + 128, aN[4], aN[5], aN[6], aN[7]);
                            const int anyb = __any_sync(FULL, bad && live);
                            if (lane == 0) wfl[q] = anyb ? 1.0 : 0.0;
                        }
#pragma unroll
                        for (int k = 0; k < 4; ++k) sP[2 * SA_FS + k * R] = make_double2(aN[2 * k], aN[2 * k + 1]);
                    }
                    // global operands of the Phi, Pi combine (needed at the end of phase 2)
                    double unP[P], unQ[P], acP[P], acQ[P];
                    if (s > 0) {
                        ldg256(prm.ACC[0] + po, acP[0], acP[1], acP[2], acP[3]);
                        ldg256(prm.ACC[0] + po + 128, acP[4], acP[5], acP[6], acP[7]);
                        ldg256(prm.ACC[1] + po, acQ[0], acQ[1], acQ[2], acQ[3]);
                        ldg256(prm.ACC[1] + po + 128, acQ[4], acQ[5], acQ[6], acQ[7]);
                        if (s < LS) {
                            ldg256(prm.UN[0] + po, unP[0], unP[1], unP[2], unP[3]);
                            ldg256(prm.UN[0] + po + 128, unP[4], unP[5], unP[6], unP[7]);
                            ldg256(prm.UN[1] + po, unQ[0], unQ[1], unQ[2], unQ[3]);
                            ldg256(prm.UN[1] + po + 128, unQ[4], unQ[5], unQ[6], unQ[7]);
                        }
                    }
                    // flux edges for the neighbour warps through shared memory (neighbour lanes: shuffles, after the wait)
                    if (lane == 0) { flo2[2 * q] = make_double2(H[0], H[1]); flo2[2 * q + 1] = make_double2(F[0], F[1]); }
                    if (lane == 31) { fhi2[2 * q] = make_double2(H[P - 2], H[P - 1]); fhi2[2 * q + 1] = make_double2(F[P - 2], F[P - 1]); }
                    const uint32_t fpar = (phs >> 3) & 1u;
                    phs ^= 8u;
                    warp_arrive(mbF);                                             // sync F: arrive

                    // ------------------------------------------------------------ between arrive and wait
                    // a4 for the interior points p in [2, P-2), which need own fluxes only: their differences go
                    // straight into the right-hand sides, in the shadow of the slowest warp's arrival
                    double tC[P];
                    ring_wait(2);
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const double2 m = slot[256 + k * 32 + lane]; tC[2 * k] = m.x; tC[2 * k + 1] = m.y; }
                    ring_next(2, j);
                    const double d4cC = K.d4c * Cl;
                    if (defer) {
#pragma unroll
                        for (int p = 0; p < P; ++p) tC[p] *= Cl;
                    }
#pragma unroll
                    for (int p = 2; p < P - 2; ++p) {
                        kP[p] = fma(d4cC, fma(8.0, H[p + 1] - H[p - 1], H[p - 2] - H[p + 2]), kP[p]);
                        kQ[p] = fma(tC[p], fma(8.0, F[p + 1] - F[p - 1], F[p - 2] - F[p + 2]), kQ[p]);
                    }
                    mbar_wait<false>(mbF, fpar);                                  // sync F: wait

                    // ------------------------------------------------------------ phase 2
                    double Hm2 = __shfl_up_sync(FULL, H[P - 2], 1), Hm1 = __shfl_up_sync(FULL, H[P - 1], 1);
                    double Fm2 = __shfl_up_sync(FULL, F[P - 2], 1), Fm1 = __shfl_up_sync(FULL, F[P - 1], 1);
                    double Hp0 = __shfl_down_sync(FULL, H[0], 1), Hp1 = __shfl_down_sync(FULL, H[1], 1);
                    double Fp0 = __shfl_down_sync(FULL, F[0], 1), Fp1 = __shfl_down_sync(FULL, F[1], 1);
                    // (the pre-pass and the first tile of the stage leave fluxes WITHOUT the factor C)
                    if (lane == 0) {
                        const double2 *src = (warp == 0) ? fpre2 + 2 * j : fhi2 + 2 * (q - 1);
                        const double2 x = src[0], y = src[1];
                        const double m = (warp == 0 && !defer) ? Cst : 1.0;
                        Hm2 = x.x * m; Hm1 = x.y * m; Fm2 = y.x * m; Fm1 = y.y * m;
                    }
                    if (lane == 31) {
                        const double2 *src = (q + 1 < NQ) ? flo2 + 2 * (q + 1) : ftop2;
                        const double2 x = src[0], y = src[1];
                        const double m = (!FIXED && after_defer && warp == SA_NW - 1) ? Cst : 1.0;     // (q + 1 is the first slice of the first tile)
                        Hp0 = x.x * m; Hp1 = x.y * m; Fp0 = y.x * m; Fp1 = y.y * m;
                    }
                    if (first) { Hm2 = H[2]; Hm1 = H[1]; Fm2 = -F[2]; Fm1 = -F[1]; }      // x=0: H even, F odd
                    if (last) {                                                   // x=pi/2: H odd with H=0 there; F even, limit of R5
                        Hp0 = 0.0; Hp1 = -H[P - 1];
                        Fp0 = Gtop * K.inv12h2; Fp1 = F[P - 1];
                    }
                    {
                        const double q0 = kQ[0];
                        kP[0] = fma(d4cC, fma(8.0, H[1] - Hm1, Hm2 - H[2]), kP[0]);
                        kQ[0] = fma(tC[0], fma(8.0, F[1] - Fm1, Fm2 - F[2]), q0);
                        kP[1] = fma(d4cC, fma(8.0, H[2] - H[0], Hm1 - H[3]), kP[1]);
                        kQ[1] = fma(tC[1], fma(8.0, F[2] - F[0], Fm1 - F[3]), kQ[1]);
                        kP[P - 2] = fma(d4cC, fma(8.0, H[P - 1] - H[P - 3], H[P - 4] - Hp0), kP[P - 2]);
                        kQ[P - 2] = fma(tC[P - 2], fma(8.0, F[P - 1] - F[P - 3], F[P - 4] - Fp0), kQ[P - 2]);
                        kP[P - 1] = fma(d4cC, fma(8.0, Hp0 - H[P - 2], H[P - 3] - Hp1), kP[P - 1]);
                        kQ[P - 1] = fma(tC[P - 1], fma(8.0, Fp0 - F[P - 2], F[P - 3] - Fp1), kQ[P - 1]);
                        if (first) {                     // Phi(0,t)=0 (eq 7); Pi_dot(0) = 3 (A e^{-delta} Phi)'(0) (R4)
                            kP[0] = 0.0;
                            kQ[0] = fma(Gorg, K.c_org * Cl, q0);
                        }
                    }
                    // a5: RK combine; at the first stage u^n is the stage state itself, still in shared memory
                    double nP[P], nQ[P];
                    if (s < LS) {
                        if (s == 0) {
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const double2 x = sP[k * R], y = sP[SA_FS + k * R];
                                unP[2 * k] = x.x; unP[2 * k + 1] = x.y; unQ[2 * k] = y.x; unQ[2 * k + 1] = y.y;
                                acP[2 * k] = x.x; acP[2 * k + 1] = x.y; acQ[2 * k] = y.x; acQ[2 * k + 1] = y.y;
                            }
                        }
#pragma unroll
                        for (int p = 0; p < P; ++p) {
                            acP[p] = fma(b_w, kP[p], acP[p]); acQ[p] = fma(b_w, kQ[p], acQ[p]);
                            nP[p] = fma(a_next, kP[p], unP[p]); nQ[p] = fma(a_next, kQ[p], unQ[p]);
                        }
                        stg256(prm.ACC[0] + po, acP[0], acP[1], acP[2], acP[3]);
                        stg256(prm.ACC[0] + po + 128, acP[4], acP[5], acP[6], acP[7]);
                        stg256(prm.ACC[1] + po, acQ[0], acQ[1], acQ[2], acQ[3]);
                        stg256(prm.ACC[1] + po + 128, acQ[4], acQ[5], acQ[6], acQ[7]);
                    } else {
#pragma unroll
                        for (int p = 0; p < P; ++p) { nP[p] = fma(b_w, kP[p], acP[p]); nQ[p] = fma(b_w, kQ[p], acQ[p]); }
                        stg256(prm.UN[0] + po, nP[0], nP[1], nP[2], nP[3]);
                        stg256(prm.UN[0] + po + 128, nP[4], nP[5], nP[6], nP[7]);
                        stg256(prm.UN[1] + po, nQ[0], nQ[1], nQ[2], nQ[3]);
                        stg256(prm.UN[1] + po + 128, nQ[4], nQ[5], nQ[6], nQ[7]);
                    }
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        sP[k * R] = make_double2(nP[2 * k], nP[2 * k + 1]);
                        sP[SA_FS + k * R] = make_double2(nQ[2 * k], nQ[2 * k + 1]);
                    }
                    // a1/a2 of the NEW stage state: thread total of f', warp-level suffix scan, slice total
                    if constexpr (!FIXED) {
                        double tot = 0.0, f7 = 0.0;
#pragma unroll
                        for (int p = 0; p < P; ++p) {
                            f7 = m2[p] * fma(nP[p], nP[p], nQ[p] * nQ[p]);
                            tot += f7;
                        }
                        if (last) tot += f7 * (1.0 / 12.0);
                        if (!live) tot = 0.0;
#pragma unroll
                        for (int d = 16; d >= 1; d >>= 1) tot += __shfl_xor_sync(FULL, tot, d);
                        if (lane == 0) wt[q] = tot;
                    }
                }   // tiles
                if (collapsed) break;
            }   // stages
            if (collapsed || n == prm.nsteps) break;
            ++n;
            if (n == prm.nsteps && !prm.check_last) break;
        }   // steps

        // ---- store the chunk in the natural layout (live points only)
        for (int j = 0; j < n_my; ++j) {
            const int q = SA_NW * j + warp, l0 = q * SA_SL + lane * P;
            const int R = sa_rs(j);
            if (l0 < npts) {
#pragma unroll
                for (int f = 0; f < (FIXED ? 2 : 3); ++f) {
                    const double2 *d = S + sa_idx(f, j, 0, tid);
                    const double2 x0 = d[0], x1 = d[R], x2 = d[2 * R], x3 = d[3 * R];
                    double *dst = prm.U[f] + row + ci0 + l0;
                    stg256(dst, x0.x, x0.y, x1.x, x1.y);
                    stg256(dst + 4, x2.x, x2.y, x3.x, x3.y);
                }
            }
        }
        if (c == 0 && tid == 0) {
            const long long sd = rec->steps_done + (long long)n;
            rec->steps_done = sd;
            if (collapsed) { rec->collapsed = 1; rec->t_collapse = (double)sd * pb.dt; }
        }
        __syncthreads();
    }   // members

    // no bulk copy may still be in flight when the CTA's shared memory is released
    if (n_my > 0) {
        if (!FIXED) ring_wait(0);
        ring_wait(1); ring_wait(2);
    }
}

// ------------------------------------------------------------------ host side
// Chunks per member G and concurrent members: every CTA of a member must be co-resident (one CTA per SM); a chunk
// is a whole number of 256-point warp slices, at most 28.  Among the feasible G the one that moves the most members
// per unit of time is taken: a stage costs one round per 8 slices plus roughly one round for the barrier.
bool stream_async_select(int N, int B, int sms, int *pG, int *pSQ, int *pgroups)
{
    if (sms <= 0 || (N - 1) % SA_P != 0) return false;
    const int nsl = (N - 1 + SA_SL - 1) / SA_SL;                    // slices per member
    const int gmin = (nsl + SA_MAXQ - 1) / SA_MAXQ;
    if (gmin > sms) return false;
    int bestG = 0, bestSQ = 0, bestGroups = 0;
    double best = -1.0;
    for (int G = gmin; G <= sms && G <= nsl; ++G) {
        const int SQ = (nsl + G - 1) / G;
        const int Ge = (nsl + SQ - 1) / SQ;                         // chunks actually needed with SQ slices each
        if (Ge != G) continue;
        int groups = sms / G;
        if (groups > B) groups = B;
        if (groups < 1 || groups * G > SP_MAX_CTAS) continue;
        const int rounds = (B + groups - 1) / groups;               // passes over the ensemble
        const double cost = (double)rounds * ((SQ + SA_NW - 1) / SA_NW + 1.0 + 0.02 * G);
        const double score = 1.0 / cost;
        if (score > best * (1.0 + 1e-9)) { best = score; bestG = G; bestSQ = SQ; bestGroups = groups; }
    }
    if (bestG == 0) return false;
    *pG = bestG; *pSQ = bestSQ; *pgroups = bestGroups;
    return true;
}

cudaError_t launch_tabp(adsc_ctx *c)
{
    const int NP = c->pb.NP;
    k_tabp<<<(NP + 255) / 256, 256, 0, c->stream>>>(c->pb.N, NP, c->tb, 1.0 / (12.0 * c->pb.h), c->ws.tabp);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_stream_async(adsc_ctx *c, long long nsteps, int check_last)
{
    const void *fn = c->pb.fixed_bg ? (const void *)k_stream_async<true> : (const void *)k_stream_async<false>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SA_SMEM);
    if (e != cudaSuccess) return e;
    // mailbox stamps count the barrier rounds of THIS launch from 1: clear what the last launch left behind
    e = cudaMemsetAsync(c->ws.sp_mbox, 0, sizeof(double) * (size_t)c->sp_groups * 2 * c->sp_G * SA_MBOX, c->stream);
    if (e != cudaSuccess) return e;
    SAParams prm;
    prm.pb = c->pb; prm.tb = c->tb;
    for (int v = 0; v < 3; ++v) { prm.U[v] = c->ws.U[v]; prm.UN[v] = c->ws.Ua[v]; prm.ACC[v] = c->ws.ACC[v]; }
    prm.tabp = c->ws.tabp;
    prm.rec = c->ws.rec; prm.mbox = c->ws.sp_mbox;
    prm.nsteps = nsteps; prm.check_last = check_last;
    prm.G = c->sp_G; prm.groups = c->sp_groups; prm.SQ = c->sp_SQ;
    {
        const double h = c->pb.h, dt = c->pb.dt, koc = c->pb.ko_eps / (64.0 * h);
        SAConsts &k = prm.k;
        k.d4c = 1.0 / (12.0 * h);
        k.kw[0] = -20.0 * koc; k.kw[1] = 15.0 * koc; k.kw[2] = -6.0 * koc; k.kw[3] = koc;
        k.hh = 0.5 * h; k.c25 = 25.0 * h / 48.0; k.c12 = 0.25 * h; k.c1 = h / 48.0;
        k.inv12h2 = 1.0 / (12.0 * h * h); k.c_org = 1.0 / (2.0 * h);
        rk_tableau(c->rk_order, dt, k.a_next, k.b_w);
        k.ns = c->rk_order;
        k.thr = c->pb.thr;
    }
    void *args[] = { (void *)&prm };
    e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)(c->sp_G * c->sp_groups)), dim3((unsigned)SA_T), args,
                                    SA_SMEM, c->stream);
    c->launches++;
    return e;
}

}  // namespace adsc
