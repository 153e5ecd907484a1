// mp_persistent_ldg.cu -- "algo 3": the whole MP loop (Eq. 8-12) as one persistent cooperative kernel whose
// correlation pass reads the dictionary straight from global memory into registers (128-bit ld.global.cg, many in
// flight per lane) instead of staging it in shared memory with TMA bulk copies (algo 1, mp_persistent.cu).
//
// Why a second streaming scheme: measured on B200, the TMA-fed kernels top out near 6.5 TB/s chip-wide whether the
// dictionary comes from HBM or from L2, while plain 128-bit loads reach 7.3 TB/s from HBM and 17-18 TB/s from L2
// (profiles/persistent_r01.md).  So this variant is what the cache-resident regime (CFG2, CFG4 <= 64 MiB) wants, and
// it removes the shared-memory staging traffic altogether: shared memory only holds the residual.
//
//   * grid = one CTA per SM (cooperative launch); CTA b owns atoms [b*M/G, (b+1)*M/G).
//   * work items = (group of A atoms, chunk of 32*UC float4 of their rows), A*UC = 16: a lane issues 16 independent
//     16-byte loads per item; (A, UC) = (2, 8) for long rows ... (16, 1) for short ones.  Items are dealt round-robin to
//     the warps, so the rounds are full whatever M/G is; the per-item partial dots go to shared memory and are added
//     per atom in ascending chunk order (deterministic), then the packed argmax (Eq. 16).
//   * one item per warp is always in flight: the first item of the next iteration is requested BEFORE the grid
//     barrier (the dictionary never changes), so the stream does not drain at the iteration boundary.
//   * everything after the dots (block argmax -> red.max.u64 -> ONE grid barrier -> Eq. 11 on the CTA's own float64
//     residual with Eq. 18 as a direct sum -> stop test) is the scheme of algo 1.
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kLdgMaxWarps = 32;

// Optional phase timeline (profiling builds only, -DMP_K1_TIMING): clock64 stamps of thread 0 of a few CTAs per iteration.
#ifdef MP_K1_TIMING
constexpr int kK1StampIters = 96, kK1StampCtas = 4, kK1StampSlots = 10;
__device__ long long g_k1_stamps[kK1StampCtas][kK1StampIters][kK1StampSlots];
#define K1_STAMP(slot)                                                                                          \
    do {                                                                                                        \
        if (tid == 0 && t < kK1StampIters && (blockIdx.x % 49) == 0 && blockIdx.x / 49 < kK1StampCtas)          \
            g_k1_stamps[blockIdx.x / 49][t][slot] = clock64();                                                  \
    } while (0)
#else
#define K1_STAMP(slot) do {} while (0)
#endif

struct LdgParams {
    const float* psi_t;
    const float* y;
    float* x;
    float* r;
    int* n_iter;
    int* idx_trace;
    float* c_trace;
    double* x64;
    unsigned long long* ctrl;   // [0] barrier counter, [1..3] rotating key slots
    int64_t ld;
    int N, M, Npad, Nr;
    float eps;
    int max_iter;
    int demote;                 // hand the pinned rows back at the end (knob l2_demote, default on)
    int resident_groups;        // groups of A atoms per CTA loaded with L2::evict_last (0 = no residency hints)
    int pin_margin;             // PP: groups at either end of a CTA's share that are never pinned
    int pingpong;               // dictionaries larger than L2: odd iterations visit the items in reverse order (see the kernel)
    int dynamic;                // long shares (the HBM-streaming regime): warps draw their work items from a counter (see the kernel)
};

__device__ __forceinline__ float4 ldg_cg4(const float4* p)
{
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// A atoms x UC float4 per lane: 16 independent 16-byte loads per lane per item.  (2, 8) for long rows, (16, 1) for short ones.
// DYN: the warps draw their work items from a shared-memory counter instead of taking every W-th one.
// PP ("ping-pong"): odd iterations visit the CTA's items in reverse order.  A dictionary larger than L2, streamed in the same order every
// iteration, gets no reuse out of an LRU cache; turned around at every iteration boundary, the rows read last are read first again, so whatever
// part of L2 is not held by the pinned rows serves the first part of every pass (cfg3: 32.3 -> 28.7 us per iteration together with a larger pinned
// set, profiles/k1_boundary_r02.md).  The order in which a CTA visits its items does not enter any result.
template <int A, int UC, bool DYN, bool PP>
__global__ void __launch_bounds__(512, 1)
mp_persistent_ldg_kernel(const LdgParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int THREADS = blockDim.x, W = THREADS >> 5;
    const int G = gridDim.x;

    double* r64 = reinterpret_cast<double*>(smem_raw);                         // Nr doubles (master residual)
    float* r32 = reinterpret_cast<float*>(r64 + p.Nr);                         // Nr floats (fp32 rounding, feeds the dots)
    unsigned long long* wkey = reinterpret_cast<unsigned long long*>(r32 + p.Nr);
    double* red = reinterpret_cast<double*>(wkey + kLdgMaxWarps);
    unsigned long long* skey = reinterpret_cast<unsigned long long*>(red + kLdgMaxWarps);
    int* next_item = reinterpret_cast<int*>(skey + 1);                          // items beyond the first W are drawn from this counter
    float* part = reinterpret_cast<float*>(skey + 2);                          // [atom of this CTA][chunk] partial dots

    if (tid < kLdgMaxWarps) red[tid] = 0.0;                                     // partial sums of absent warps stay 0
    if (tid == 0) *next_item = THREADS >> 5;
    __syncthreads();
    const int a0 = (int)(((int64_t)blockIdx.x * p.M) / G);
    const int a1 = (int)(((int64_t)(blockIdx.x + 1) * p.M) / G);
    const int n_atoms = a1 - a0;
    const int n_groups = (n_atoms + A - 1) / A;
    const int n4 = p.Npad >> 2;
    const int n_chunks = (n4 + 32 * UC - 1) / (32 * UC);
    const int n_items = n_groups * n_chunks;
    const bool ragged = p.Npad != p.N;

    // ---- Eq. 8: r <- y (float64 master + fp32 copy), ||y||^2 -------------------------------------------------------
    double ss = 0.0;
    for (int n = tid; n < p.Nr; n += THREADS) {
        const float v = n < p.N ? p.y[n] : 0.f;
        r64[n] = (double)v;
        r32[n] = v;
        ss += (double)v * (double)v;
    }
    ss = warp_sum(ss);
    if (lane == 0) red[warp] = ss;
    __syncthreads();
    double rr = 0.0;
    for (int w = 0; w < W; w++) rr += red[w];
    const double thresh2 = ((double)p.eps * (double)p.eps) * rr;                // ||r|| > eps ||y||  <=>  ||r||^2 > eps^2 ||y||^2
    __syncthreads();

    const float4* r4 = reinterpret_cast<const float4*>(r32);
    const uint64_t pol_last = l2_policy_evict_last(), pol_first = l2_policy_evict_first();
    float4 v[A][UC];
    // pinned groups: spread evenly over the share, or (PP) over its middle only -- the p.pin_margin groups at either end are the ones the
    // reversed order re-reads soonest, they are served by recency and need no pin
    auto group_is_pinned = [&](int g) {
        const int e = PP ? p.pin_margin : 0;
        return g >= e && g < n_groups - e && l2_group_is_resident(g - e, p.resident_groups, n_groups - 2 * e);
    };
    auto load_item = [&](int item, bool flip) {
        if (flip) item = n_items - 1 - item;
        const int g = item / n_chunks, ch = item - g * n_chunks;
        const int jb = ch * 32 * UC + lane;
        if (A <= 4 && p.resident_groups > 0) {                                  // dictionary larger than L2: residency hints (long rows only:
                                                                                // the short-row variants have no registers to spare)
            // The resident groups are spread evenly over the CTA's share (Bresenham), so that L2 hits and HBM misses
            // interleave in time: with the resident rows first, HBM idled while every CTA read them (35.4 -> 33.3 us).
            const uint64_t pol = group_is_pinned(g) ? pol_last : pol_first;
#pragma unroll
            for (int a = 0; a < A; a++) {
                const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;
                const float4* row = reinterpret_cast<const float4*>(p.psi_t + (int64_t)(a0 + rel) * p.ld);
#pragma unroll
                for (int u = 0; u < UC; u++) {
                    const int j = jb + 32 * u;
                    v[a][u] = j < n4 ? ldg_cg4_hint(row + j, pol) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
            return;
        }
#pragma unroll
        for (int a = 0; a < A; a++) {
            const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;      // a short last group re-reads its last atom
            const float4* row = reinterpret_cast<const float4*>(p.psi_t + (int64_t)(a0 + rel) * p.ld);
#pragma unroll
            for (int u = 0; u < UC; u++) {
                const int j = jb + 32 * u;
                v[a][u] = j < n4 ? ldg_cg4(row + j) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
    };
    int it = warp;
    bool have = it < n_items;
    if (have) load_item(it, false);
    int t = 0;
    // ---- the loop: while ||r|| > eps ||y|| and t < T -----------------------------------------------------------
    while ((rr > thresh2) && (t < p.max_iter)) {
        K1_STAMP(0);
        // ---------- Eq. 9: items = (group of A atoms, chunk of 32*UC float4).  Warp w starts with item w; when the share is long
        // (DYN: the HBM-streaming regime) every further item is drawn from a shared-memory counter: a warp whose rows came from L2
        // (resident groups) or from a faster HBM channel takes more items, so the CTA is done when its share is done, not when its
        // unluckiest warp is (profiles/k1_boundary_r02.md: the warps of one CTA finished up to 3 400 cycles apart).
        // An atom's dot product is the same arithmetic whichever warp computes it, so the results do not depend on the dealing.
        // One item is always in flight per warp: `v` was loaded before the previous iteration's barrier (or in the
        // prologue), so the stream does not drain while the CTAs meet and update the residual.
        while (have) {
            int nxt = it + W;                                                   // short shares (< 8 items per warp): plain round-robin
            if (DYN && lane == 0) nxt = atomicAdd(next_item, 1);
            const bool flip = PP && (t & 1);
            const int itm = flip ? n_items - 1 - it : it;
            const int g = itm / n_chunks, ch = itm - g * n_chunks;
            const int atom0 = g * A;                                           // relative to a0
            const int jb = ch * 32 * UC + lane;
            float acc[A];
#pragma unroll
            for (int a = 0; a < A; a++) acc[a] = 0.f;
#pragma unroll
            for (int u = 0; u < UC; u++) {
                const int j = jb + 32 * u;
                float4 rv = j < n4 ? r4[j] : make_float4(0.f, 0.f, 0.f, 0.f);
                if (ragged && j == n4 - 1) {                                   // N % 4 != 0: up to 3 caller-owned pad floats per row
                    const int n = j << 2;
#pragma unroll
                    for (int a = 0; a < A; a++) {
                        if (n + 1 >= p.N) v[a][u].y = 0.f;
                        if (n + 2 >= p.N) v[a][u].z = 0.f;
                        v[a][u].w = 0.f;
                    }
                }
#pragma unroll
                for (int a = 0; a < A; a++) {
                    acc[a] = fmaf(v[a][u].x, rv.x, acc[a]); acc[a] = fmaf(v[a][u].y, rv.y, acc[a]);
                    acc[a] = fmaf(v[a][u].z, rv.z, acc[a]); acc[a] = fmaf(v[a][u].w, rv.w, acc[a]);
                }
            }
            it = DYN ? __shfl_sync(0xffffffffu, nxt, 0) : nxt;
            have = it < n_items;
            if (have) load_item(it, flip);
#pragma unroll
            for (int a = 0; a < A; a++) {
                const float c = warp_sum(acc[a]);
                if (lane == a && atom0 + a < n_atoms) part[(atom0 + a) * n_chunks + ch] = c;
            }
        }
        it = warp;                                                             // the dictionary never changes: the first item of
        have = it < n_items;                                                   // the next iteration is requested ahead of the barrier
        if (have) load_item(it, PP && ((t + 1) & 1));
        K1_STAMP(1);
        __syncthreads();
        if (DYN && tid == 0) *next_item = W;                                   // nobody draws again before the next barriers
        K1_STAMP(2);
        // ---------- Eq. 9 finished per atom (chunks added in ascending order), Eq. 16 packed argmax ----------------------
        unsigned long long best = 0ull;
        for (int a = tid; a < n_atoms; a += THREADS) {
            float c = part[a * n_chunks];
            for (int ch = 1; ch < n_chunks; ch++) c += part[a * n_chunks + ch];
            const unsigned long long k = pack_key(c, a0 + a);
            best = k > best ? k : best;
        }
        best = warp_max_redux(best);

        // ---------- block argmax -> grid argmax, ONE grid barrier (mp_common.cuh) ---------------------------------------------
        K1_STAMP(3);
#ifdef MP_K1_TIMING
        long long st_arrive = 0, st_done = 0;
        const unsigned long long key = grid_argmax(best, wkey, skey, p.ctrl, t, &st_arrive, &st_done);
        if (tid == 0 && t < kK1StampIters && (blockIdx.x % 49) == 0 && blockIdx.x / 49 < kK1StampCtas) {
            g_k1_stamps[blockIdx.x / 49][t][4] = st_arrive; g_k1_stamps[blockIdx.x / 49][t][5] = st_done;
        }
#else
        const unsigned long long key = grid_argmax(best, wkey, skey, p.ctrl, t);
#endif
        K1_STAMP(6);
        const int i = key_index(key);
        const float c = key_value(key);
        const double cd = (double)c;

        // ---------- Eq. 11 on this CTA's float64 r, Eq. 18 direct sum ------------------------------------------------
        {
            const float4* psi4 = reinterpret_cast<const float4*>(p.psi_t + (int64_t)i * p.ld);
            double s2 = 0.0;
            for (int j = tid; j < n4; j += THREADS) {
                const float4 q = __ldg(psi4 + j);
                const int n = j << 2;
                double v0 = r64[n] - cd * (double)q.x;
                double v1 = r64[n + 1] - cd * (double)q.y;
                double v2 = r64[n + 2] - cd * (double)q.z;
                double v3 = r64[n + 3] - cd * (double)q.w;
                if (n + 3 >= p.N) {                                             // keep the pad of r at zero
                    if (n + 1 >= p.N) v1 = 0.0;
                    if (n + 2 >= p.N) v2 = 0.0;
                    v3 = 0.0;
                }
                r64[n] = v0; r64[n + 1] = v1; r64[n + 2] = v2; r64[n + 3] = v3;
                *reinterpret_cast<float4*>(r32 + n) = make_float4((float)v0, (float)v1, (float)v2, (float)v3);
                s2 += v0 * v0; s2 += v1 * v1; s2 += v2 * v2; s2 += v3 * v3;
            }
            K1_STAMP(7);
            s2 = warp_sum(s2);
            if (lane == 0) red[warp] = s2;
        }
        // ---------- Eq. 10, Eq. 12, traces: CTA 0 only ---------------------------------------------------------------
        if (blockIdx.x == 0 && tid == THREADS - 32) {                          // not the thread every CTA's barrier waits for
            record_step(p.x64, p.idx_trace, p.c_trace, p.ctrl, t, i, c);
        }
        __syncthreads();
        {                                                                       // W <= 16 partials (absent warps hold 0), fixed tree
            const double2* r2 = reinterpret_cast<const double2*>(red);
            const double2 q0 = r2[0], q1 = r2[1], q2 = r2[2], q3 = r2[3], q4 = r2[4], q5 = r2[5], q6 = r2[6], q7 = r2[7];
            rr = (((q0.x + q0.y) + (q1.x + q1.y)) + ((q2.x + q2.y) + (q3.x + q3.y))) +
                 (((q4.x + q4.y) + (q5.x + q5.y)) + ((q6.x + q6.y) + (q7.x + q7.y)));
        }
        K1_STAMP(8);
        t += 1;
    }

    // ---- hand the pinned rows back to the L2's normal replacement (see l2_demote_row) ------------------------------------------
    if (A <= 4 && p.resident_groups > 0 && p.demote) {
        for (int g = warp; g < n_groups; g += W) {
            if (!group_is_pinned(g)) continue;
            for (int a = 0; a < A; a++) {
                const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;
                l2_demote_row(p.psi_t + (int64_t)(a0 + rel) * p.ld, (size_t)p.Npad * 4, lane);
            }
        }
    }
    // ---- P:86 return x~ (and r, t): CTA 0 -------------------------------------------------------------------------------
    if (blockIdx.x == 0) {
        __threadfence();                                                        // the x~ accumulations of this CTA (thread THREADS - 32)
        __syncthreads();
        for (int m = tid; m < p.M; m += THREADS) p.x[m] = (float)__ldcg(p.x64 + m);
        for (int n = tid; n < p.N; n += THREADS) p.r[n] = r32[n];
        if (tid == 0) *p.n_iter = t;
    }
}

// ------------------------------------------------------------------------------------------------------------------
struct LdgPlan {
    int A, UC, W, grid, dynamic;
    size_t smem;
};

static bool ldg_plan(int N, int M, const DeviceInfo& di, LdgPlan* plan)
{
    const int n4 = round_up(N, 4) / 4;
    int A = 2, UC = 8;
    if (n4 <= 32) { A = 16; UC = 1; }
    else if (n4 <= 64) { A = 8; UC = 2; }
    else if (n4 <= 128) { A = 4; UC = 4; }
    int G = di.sm_count > 0 ? di.sm_count : 1;
    if (options().grid > 0 && options().grid < G) G = (int)options().grid;      // the knob: fewer CTAs, each with a larger share
    const int atoms_max = (M + G - 1) / G;
    const int n_chunks = (n4 + 32 * UC - 1) / (32 * UC);
    const int items = ((atoms_max + A - 1) / A) * n_chunks;
    const size_t Nr = (size_t)round_up(N, 128);
    const size_t smem = Nr * 12 + 8 * (2 * kLdgMaxWarps + 4) + 4 * (size_t)atoms_max * n_chunks + 64;
    if (smem > (size_t)di.smem_optin) return false;
    // long shares (>= 8 items per warp with 16 warps: the HBM-streaming regime): the warps draw items from a counter (knob "balance" = 1: off)
    const bool dynamic = items >= 8 * 16 && options().balance != 1;
    // warps: the fullest rounds (see mp_persistent.cu make_plan); 8..16 warps, ties to more warps
    int W = 16;
    if (options().warps >= 1 && options().warps <= 16) W = (int)options().warps;
    else if (!dynamic) {                                                        // dynamic dealing needs no full rounds
        double best = -1.0;
        for (int w = 8; w <= 16; w++) {
            const double fill = (double)items / ((double)((items + w - 1) / w) * w);
            if (fill >= best) { best = fill; W = w; }
        }
    }
    plan->A = A; plan->UC = UC; plan->W = W; plan->smem = smem;
    plan->grid = G; plan->dynamic = dynamic ? 1 : 0;
    return true;
}

bool persistent_ldg_supported(int N, int M)
{
    DeviceInfo di;
    if (device_info(&di) != MP_OK || !di.coop) return false;
    LdgPlan plan;
    return ldg_plan(N, M, di, &plan);
}

template <int A, int UC, bool DYN, bool PP>
static mp_status launch_ldg_mode(const LdgParams& p, const LdgPlan& plan, int device, cudaStream_t stream)
{
    static thread_local int attr_dev = -1;
    if (attr_dev != device) {
        MP_CUDA(cudaFuncSetAttribute(mp_persistent_ldg_kernel<A, UC, DYN, PP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        attr_dev = device;
    }
    int occ = 0;
    MP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mp_persistent_ldg_kernel<A, UC, DYN, PP>, plan.W * 32, plan.smem));
    if (occ < 1) return fail(MP_ERR_UNSUPPORTED, "register-streaming persistent kernel does not fit one CTA per SM");
    void* args[] = {(void*)&p};
    MP_CUDA(cudaLaunchCooperativeKernel((const void*)mp_persistent_ldg_kernel<A, UC, DYN, PP>, dim3(plan.grid), dim3(plan.W * 32), args,
                                        plan.smem, stream));
    count_launch();
    return MP_OK;
}
template <int A, int UC>
static mp_status launch_ldg(const LdgParams& p, const LdgPlan& plan, int device, cudaStream_t stream)
{
    if (p.dynamic) return p.pingpong ? launch_ldg_mode<A, UC, true, true>(p, plan, device, stream) : launch_ldg_mode<A, UC, true, false>(p, plan, device, stream);
    return p.pingpong ? launch_ldg_mode<A, UC, false, true>(p, plan, device, stream) : launch_ldg_mode<A, UC, false, false>(p, plan, device, stream);
}

mp_status launch_recover_persistent_ldg(const RecoverArgs& a, const Workspace& ws, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    if (!di.coop) return fail(MP_ERR_UNSUPPORTED, "device does not support cooperative launch");
    LdgPlan plan;
    if (!ldg_plan(a.N, a.M, di, &plan)) return fail(MP_ERR_UNSUPPORTED, "N=%d, M=%d do not fit the register-streaming kernel's shared memory", a.N, a.M);

    MP_CUDA(cudaMemsetAsync(ws.ctrl, 0, 256 + sizeof(double) * (size_t)a.M, stream));
    LdgParams p;
    p.psi_t = a.psi_t; p.y = a.y; p.x = a.x; p.r = a.r; p.n_iter = a.n_iter;
    p.idx_trace = a.idx_trace; p.c_trace = a.c_trace;
    p.x64 = ws.x64; p.ctrl = ws.ctrl; p.ld = a.ld;
    p.N = a.N; p.M = a.M; p.Npad = round_up(a.N, 4); p.Nr = round_up(a.N, 128);
    p.eps = a.eps; p.max_iter = a.max_iter;
    // L2 residency: only for dictionaries that do not fit in L2 anyway.  Knob "l2_resident_mb": 0 = auto (68 MB), 1 = off.
    p.demote = options().l2_demote != 1;
    const L2Plan l2 = l2_plan(4.0 * (double)a.ld * a.M, plan.grid, 4.0 * (double)a.ld * plan.A,
                              ((a.M + plan.grid - 1) / plan.grid + plan.A - 1) / plan.A, true);
    p.pingpong = l2.pingpong; p.resident_groups = l2.resident_groups; p.pin_margin = l2.pin_margin;
    p.dynamic = plan.dynamic;
    options().info_l2_pingpong = p.pingpong; options().info_l2_dynamic = p.dynamic;
    options().info_l2_resident_mb = (int64_t)((double)p.resident_groups * plan.grid * 4.0 * (double)a.ld * plan.A / 1e6 + 0.5);
    if (plan.A == 16) return launch_ldg<16, 1>(p, plan, di.device, stream);
    if (plan.A == 8) return launch_ldg<8, 2>(p, plan, di.device, stream);
    if (plan.A == 4) return launch_ldg<4, 4>(p, plan, di.device, stream);
    return launch_ldg<2, 8>(p, plan, di.device, stream);
}

}  // namespace mp

#ifdef MP_K1_TIMING
extern "C" __attribute__((visibility("default"))) int mp_debug_k1_stamps(long long* out, size_t bytes)
{
    if (bytes > sizeof(mp::g_k1_stamps)) bytes = sizeof(mp::g_k1_stamps);
    return (int)cudaMemcpyFromSymbol(out, mp::g_k1_stamps, bytes);
}
#endif
