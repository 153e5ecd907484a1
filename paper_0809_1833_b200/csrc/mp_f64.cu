// mp_f64.cu -- the double-precision path (the paper reports single AND double precision, P:131-158,
// P:171): column normalisation and the whole MP loop (Eq. 8-12) on a float64 dictionary.
//
// Same scheme as the register-streaming fp32 kernel (mp_persistent_ldg.cu): one persistent cooperative kernel, one CTA
// per SM, work items = (group of A atoms, chunk of 32*UC 16-byte vectors) streamed from global memory into registers,
// one item per warp in flight across the iteration boundary, one grid barrier per iteration, residual replicated per CTA.
// What differs: everything is float64 (dots, residual, norms); a 64-bit packed key cannot hold a float64 magnitude and
// an index, so every CTA publishes its best (c, index) pair to its own slot before the barrier and every CTA scans the G
// slots after it (same total order everywhere: larger |c|, then smaller index; NaN never wins).
// Roofline: HBM, 8NM bytes per iteration -- half the iterations/s of the fp32 path at the same N, M.
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kF64MaxWarps = 32;
constexpr int kF64Slots = 1024;          // >= CTAs of the grid

struct Cand {                            // a candidate of the argmax: signed correlation and atom index
    double c;
    int idx, pad;
};

struct F64Params {
    const double* psi_t;
    const double* y;
    double* x;
    double* r;
    int* n_iter;
    int* idx_trace;
    double* c_trace;
    double* xacc;               // M accumulators (zeroed by the launcher)
    unsigned long long* ctrl;   // [0] barrier counter
    Cand* slots;                // [2][kF64Slots]
    int64_t ld;
    int N, M, Npad, Nr;         // Npad = N rounded up to 2, Nr = N rounded up to 128
    double eps;
    int max_iter;
    int demote;                 // hand the pinned rows back at the end (knob l2_demote, default on)
    int resident_groups;        // groups of A atoms per CTA loaded L2::evict_last (mp_common.cuh), 0 = no hints
    int pingpong, pin_margin;   // DYN kernels: reversed item order on odd iterations, unpinned groups at either end (mp_internal.h l2_plan)
};

__device__ __forceinline__ double2 ldg_cg_d2(const double2* p)
{
    double2 v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double abs_or_minus1(double c) { return c == c ? fabs(c) : -1.0; }      // NaN never wins (R2)
__device__ __forceinline__ bool cand_better(double ca, int ia, double cb, int ib)
{
    const double a = abs_or_minus1(ca), b = abs_or_minus1(cb);
    return a > b || (a == b && ia < ib);
}
__device__ __forceinline__ void warp_best(double& c, int& idx)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double oc = __shfl_xor_sync(0xffffffffu, c, o);
        const int oi = __shfl_xor_sync(0xffffffffu, idx, o);
        if (cand_better(oc, oi, c, idx)) { c = oc; idx = oi; }
    }
}

// DYN (long shares, the HBM-streaming regime): warps draw their work items from a shared-memory counter, as in mp_persistent_ldg.cu
template <int A, int UC, bool DYN>
__global__ void __launch_bounds__(512, 1)
mp_persistent_f64_kernel(const F64Params p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int THREADS = blockDim.x, W = THREADS >> 5;
    const int G = gridDim.x;
    constexpr int kNoAtom = 0x7FFFFFFF;

    double* rres = reinterpret_cast<double*>(smem_raw);                        // Nr doubles: the residual
    double* red = rres + p.Nr;                                                 // W
    double* wc = red + kF64MaxWarps;                                           // W   per-warp best c
    int* wi = reinterpret_cast<int*>(wc + kF64MaxWarps);                       // W   per-warp best index
    Cand* win = reinterpret_cast<Cand*>(wi + kF64MaxWarps);                    // 1   the winner of this iteration
    int* next_item = reinterpret_cast<int*>(win + 1);                          // DYN: items beyond the first W are drawn from this counter
    double* part = reinterpret_cast<double*>(next_item + 2);                   // [atom of this CTA][chunk] partial dots

    const int a0 = (int)(((int64_t)blockIdx.x * p.M) / G);
    const int a1 = (int)(((int64_t)(blockIdx.x + 1) * p.M) / G);
    const int n_atoms = a1 - a0;
    const int n_groups = (n_atoms + A - 1) / A;
    const int n2 = p.Npad >> 1;
    const int n_chunks = (n2 + 32 * UC - 1) / (32 * UC);
    const int n_items = n_groups * n_chunks;
    const bool ragged = p.Npad != p.N;

    // ---- Eq. 8: r <- y, ||y||^2 ---------------------------------------------------------------------------------------
    double ss = 0.0;
    for (int n = tid; n < p.Nr; n += THREADS) {
        const double v = n < p.N ? p.y[n] : 0.0;
        rres[n] = v;
        ss += v * v;
    }
    ss = warp_sum(ss);
    if (lane == 0) red[warp] = ss;
    __syncthreads();
    double rr = 0.0;
    for (int w = 0; w < W; w++) rr += red[w];
    const double thresh = p.eps * sqrt(rr);
    __syncthreads();

    const double2* r2 = reinterpret_cast<const double2*>(rres);
    double2 v[A][UC];
    const uint64_t pol_last = l2_policy_evict_last(), pol_first = l2_policy_evict_first();
    auto group_is_pinned = [&](int g) {
        const int e = DYN ? p.pin_margin : 0;
        return g >= e && g < n_groups - e && l2_group_is_resident(g - e, p.resident_groups, n_groups - 2 * e);
    };
    auto load_item = [&](int item, bool flip) {
        if (flip) item = n_items - 1 - item;
        const int g = item / n_chunks, ch = item - g * n_chunks;
        const int jb = ch * 32 * UC + lane;
        if (A <= 4 && p.resident_groups > 0) {                                  // dictionary larger than L2: residency hints (long rows only:
                                                                                // the short-row variants have no registers to spare)
            const uint64_t pol = group_is_pinned(g) ? pol_last : pol_first;
#pragma unroll
            for (int a = 0; a < A; a++) {
                const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;
                const double2* row = reinterpret_cast<const double2*>(p.psi_t + (int64_t)(a0 + rel) * p.ld);
#pragma unroll
                for (int u = 0; u < UC; u++) {
                    const int j = jb + 32 * u;
                    v[a][u] = j < n2 ? ldg_cg_d2_hint(row + j, pol) : make_double2(0.0, 0.0);
                }
            }
            return;
        }
#pragma unroll
        for (int a = 0; a < A; a++) {
            const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;      // a short last group re-reads its last atom
            const double2* row = reinterpret_cast<const double2*>(p.psi_t + (int64_t)(a0 + rel) * p.ld);
#pragma unroll
            for (int u = 0; u < UC; u++) {
                const int j = jb + 32 * u;
                v[a][u] = j < n2 ? ldg_cg_d2(row + j) : make_double2(0.0, 0.0);
            }
        }
    };
    int it = warp;
    bool have = it < n_items;
    if (have) load_item(it, false);
    if (DYN && tid == 0) *next_item = W;
    __syncthreads();
    int t = 0;
    // ---- the loop: while ||r|| > eps ||y|| and t < T -----------------------------------------------------------
    while ((sqrt(rr) > thresh) && (t < p.max_iter)) {
        // ---------- Eq. 9: items dealt round-robin to the warps (DYN: drawn from a counter), one always in flight -----------
        while (have) {
            int nxt = it + W;
            if (DYN && lane == 0) nxt = atomicAdd(next_item, 1);
            const bool flip = DYN && p.pingpong && (t & 1);                    // odd iterations visit the items in reverse order (mp_persistent_ldg.cu)
            const int itm = flip ? n_items - 1 - it : it;
            const int g = itm / n_chunks, ch = itm - g * n_chunks;
            const int atom0 = g * A;
            const int jb = ch * 32 * UC + lane;
            double acc[A];
#pragma unroll
            for (int a = 0; a < A; a++) acc[a] = 0.0;
#pragma unroll
            for (int u = 0; u < UC; u++) {
                const int j = jb + 32 * u;
                const double2 rv = j < n2 ? r2[j] : make_double2(0.0, 0.0);
                if (ragged && j == n2 - 1) {                                   // N odd: one caller-owned pad double per row
#pragma unroll
                    for (int a = 0; a < A; a++) v[a][u].y = 0.0;
                }
#pragma unroll
                for (int a = 0; a < A; a++) {
                    acc[a] = fma(v[a][u].x, rv.x, acc[a]);
                    acc[a] = fma(v[a][u].y, rv.y, acc[a]);
                }
            }
            it = DYN ? __shfl_sync(0xffffffffu, nxt, 0) : nxt;
            have = it < n_items;
            if (have) load_item(it, flip);
#pragma unroll
            for (int a = 0; a < A; a++) {
                const double c = warp_sum(acc[a]);
                if (lane == a && atom0 + a < n_atoms) part[(atom0 + a) * n_chunks + ch] = c;
            }
        }
        it = warp;                                                             // the dictionary never changes: first item of the
        have = it < n_items;                                                   // next iteration requested ahead of the barrier
        if (have) load_item(it, DYN && p.pingpong && ((t + 1) & 1));
        __syncthreads();
        if (DYN && tid == 0) *next_item = W;                                   // nobody draws again before the next barriers
        // ---------- Eq. 9 finished per atom (chunks in ascending order), Eq. 16 -------------------------------------------
        double bc = 0.0;
        int bi = kNoAtom;
        for (int a = tid; a < n_atoms; a += THREADS) {
            double c = part[a * n_chunks];
            for (int ch = 1; ch < n_chunks; ch++) c += part[a * n_chunks + ch];
            if (cand_better(c, a0 + a, bc, bi)) { bc = c; bi = a0 + a; }
        }
        if (bi == kNoAtom) bc = __longlong_as_double(0x7FF8000000000000ll);    // no atom: NaN loses every comparison
        warp_best(bc, bi);
        if (lane == 0) { wc[warp] = bc; wi[warp] = bi; }
        __syncthreads();
        // ---------- publish this CTA's candidate, ONE grid barrier, then everybody scans the G candidates ------------------
        if (warp == 0) {
            double c = lane < W ? wc[lane] : __longlong_as_double(0x7FF8000000000000ll);
            int i = lane < W ? wi[lane] : kNoAtom;
            warp_best(c, i);
            Cand* set = p.slots + (size_t)(t & 1) * kF64Slots;
            if (lane == 0) {
                set[blockIdx.x].c = c;
                set[blockIdx.x].idx = i;
                red_add_release_u64(p.ctrl, 1ull);
                const unsigned long long target = (unsigned long long)(t + 1) * (unsigned long long)G;
                while (ld_acquire_u64(p.ctrl) < target) {}
            }
            __syncwarp();
            double gc = __longlong_as_double(0x7FF8000000000000ll);
            int gi = kNoAtom;
            for (int s = lane; s < G; s += 32) {
                const double sc = __ldcg(&set[s].c);
                const int si = __ldcg(&set[s].idx);
                if (cand_better(sc, si, gc, gi)) { gc = sc; gi = si; }
            }
            warp_best(gc, gi);
            if (lane == 0) { win->c = gc; win->idx = gi; }
        }
        __syncthreads();
        const int i = win->idx;
        const double c = win->c;

        // ---------- Eq. 11 on this CTA's r, Eq. 18 direct sum ----------------------------------------------------------------
        {
            const double* psi_i = p.psi_t + (int64_t)i * p.ld;
            double s2 = 0.0;
            for (int n = tid; n < p.N; n += THREADS) {
                const double vn = rres[n] - c * __ldg(psi_i + n);
                rres[n] = vn;
                s2 += vn * vn;
            }
            s2 = warp_sum(s2);
            if (lane == 0) red[warp] = s2;
        }
        // ---------- Eq. 10, Eq. 12, traces: CTA 0 only -----------------------------------------------------------------------
        if (blockIdx.x == 0 && tid == 0) {
            red_add_f64(p.xacc + i, c);
            if (p.idx_trace) p.idx_trace[t] = i;
            if (p.c_trace) p.c_trace[t] = c;
        }
        __syncthreads();
        rr = 0.0;
        for (int w = 0; w < W; w++) rr += red[w];
        t += 1;
    }

    // ---- hand the pinned rows back to the L2's normal replacement (see l2_demote_row) ------------------------------------------
    if (A <= 4 && p.resident_groups > 0 && p.demote) {
        for (int g = warp; g < n_groups; g += W) {
            if (!group_is_pinned(g)) continue;
            for (int a = 0; a < A; a++) {
                const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;
                l2_demote_row(p.psi_t + (int64_t)(a0 + rel) * p.ld, (size_t)p.Npad * 8, lane);
            }
        }
    }
    // ---- P:86 return x~ (and r, t): CTA 0 -------------------------------------------------------------------------------
    if (blockIdx.x == 0) {
        if (tid == 0) __threadfence();
        __syncthreads();
        for (int m = tid; m < p.M; m += THREADS) p.x[m] = __ldcg(p.xacc + m);
        for (int n = tid; n < p.N; n += THREADS) p.r[n] = rres[n];
        if (tid == 0) *p.n_iter = t;
    }
}

// Eq. 4 in float64: one warp per atom, two passes over the row.
__global__ void __launch_bounds__(256)
normalize_columns_f64_kernel(double* __restrict__ psi_t, int N, int M, int64_t ld, double* __restrict__ norms_out)
{
    const int lane = threadIdx.x & 31;
    const int m = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (m >= M) return;
    double* row = psi_t + (int64_t)m * ld;
    double s = 0.0;
    for (int n = lane; n < N; n += 32) s += row[n] * row[n];
    s = warp_sum(s);
    const double nrm = sqrt(s);
    if (lane == 0 && norms_out) norms_out[m] = nrm;
    if (nrm > 0.0)
        for (int n = lane; n < N; n += 32) row[n] = row[n] / nrm;
}

// ------------------------------------------------------------------------------------------------------------------
struct F64Plan {
    int A, UC, W, grid; bool dynamic;
    size_t smem;
};

static bool f64_plan(int N, int M, const DeviceInfo& di, F64Plan* plan)
{
    const int n2 = round_up(N, 2) / 2;
    int A = 2, UC = 8;
    if (n2 <= 32) { A = 16; UC = 1; }
    else if (n2 <= 64) { A = 8; UC = 2; }
    else if (n2 <= 128) { A = 4; UC = 4; }
    int G = di.sm_count > 0 ? di.sm_count : 1;
    if (options().grid > 0 && options().grid < G) G = (int)options().grid;      // the knob: fewer CTAs, each with a larger share
    if (G > kF64Slots) return false;
    const int atoms_max = (M + G - 1) / G;
    const int n_chunks = (n2 + 32 * UC - 1) / (32 * UC);
    const int items = ((atoms_max + A - 1) / A) * n_chunks;
    const size_t Nr = (size_t)round_up(N, 128);
    const size_t smem = Nr * 8 + 8 * 2 * kF64MaxWarps + 4 * kF64MaxWarps + sizeof(Cand) + 8 * (size_t)atoms_max * n_chunks + 64;
    if (smem > (size_t)di.smem_optin) return false;
    int W = 16;
    if (options().warps >= 1 && options().warps <= 16) W = (int)options().warps;
    else {
        double best = -1.0;
        for (int w = 8; w <= 16; w++) {
            const double fill = (double)items / ((double)((items + w - 1) / w) * w);
            if (fill >= best) { best = fill; W = w; }
        }
    }
    plan->A = A; plan->UC = UC; plan->W = W; plan->smem = smem;
    plan->grid = G;
    plan->dynamic = A == 2 && items >= 8 * 16 && options().balance != 1;         // long shares: see mp_persistent_ldg.cu
    if (plan->dynamic && !(options().warps >= 1 && options().warps <= 16)) plan->W = 16;
    return true;
}

static size_t f64_workspace(int M) { return 256 + (sizeof(double) * (size_t)M + 255) / 256 * 256 + sizeof(Cand) * 2 * kF64Slots; }

template <int A, int UC, bool DYN = false>
static mp_status launch_f64(const F64Params& p, const F64Plan& plan, int device, cudaStream_t stream)
{
    static thread_local int attr_dev = -1;
    if (attr_dev != device) {
        MP_CUDA(cudaFuncSetAttribute(mp_persistent_f64_kernel<A, UC, DYN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        attr_dev = device;
    }
    int occ = 0;
    MP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mp_persistent_f64_kernel<A, UC, DYN>, plan.W * 32, plan.smem));
    if (occ < 1) return fail(MP_ERR_UNSUPPORTED, "float64 persistent kernel does not fit one CTA per SM");
    void* args[] = {(void*)&p};
    MP_CUDA(cudaLaunchCooperativeKernel((const void*)mp_persistent_f64_kernel<A, UC, DYN>, dim3(plan.grid), dim3(plan.W * 32), args,
                                        plan.smem, stream));
    count_launch();
    return MP_OK;
}

}  // namespace mp

using namespace mp;

extern "C" {

MP_API size_t mp_workspace_bytes_f64(int N, int M)
{
    if (N < 1 || M < 1) return 0;
    return f64_workspace(M);
}

MP_API mp_status mp_normalize_columns_f64(double* psi_t, int N, int M, int64_t ld, double* norms_out, void* stream)
{
    if (!psi_t) return fail(MP_ERR_INVALID_ARG, "psi_t is null");
    if (N < 1 || M < 1 || ld < N) return fail(MP_ERR_INVALID_ARG, "need N >= 1, M >= 1, ld >= N");
    normalize_columns_f64_kernel<<<(M + 7) / 8, 256, 0, static_cast<cudaStream_t>(stream)>>>(psi_t, N, M, ld, norms_out);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

MP_API mp_status mp_recover_f64(const double* psi_t, int N, int M, int64_t ld,
                                const double* y, double eps, int max_iter,
                                double* x, double* r, int* n_iter,
                                int* idx_trace, double* c_trace,
                                void* workspace, size_t workspace_bytes, void* stream)
{
    if (!psi_t || !y || !x || !r || !n_iter) return fail(MP_ERR_INVALID_ARG, "psi_t, y, x, r and n_iter must be non-null");
    if (N < 1 || M < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1 and M >= 1 (got N=%d, M=%d)", N, M);
    if (ld < N || (ld & 1)) return fail(MP_ERR_INVALID_ARG, "need ld >= N and ld %% 2 == 0 (got ld=%lld, N=%d)", (long long)ld, N);
    if (reinterpret_cast<uintptr_t>(psi_t) & 15u) return fail(MP_ERR_INVALID_ARG, "psi_t must be 16-byte aligned");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    const size_t need = f64_workspace(M);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    if (!di.coop) return fail(MP_ERR_UNSUPPORTED, "device does not support cooperative launch");
    F64Plan plan;
    if (!f64_plan(N, M, di, &plan)) return fail(MP_ERR_UNSUPPORTED, "N=%d, M=%d do not fit the float64 kernel's shared memory", N, M);

    cudaStream_t s = static_cast<cudaStream_t>(stream);
    char* base = static_cast<char*>(workspace);
    MP_CUDA(cudaMemsetAsync(base, 0, need, s));
    F64Params p;
    p.psi_t = psi_t; p.y = y; p.x = x; p.r = r; p.n_iter = n_iter; p.idx_trace = idx_trace; p.c_trace = c_trace;
    p.ctrl = reinterpret_cast<unsigned long long*>(base);
    p.xacc = reinterpret_cast<double*>(base + 256);
    p.slots = reinterpret_cast<Cand*>(base + 256 + (sizeof(double) * (size_t)M + 255) / 256 * 256);
    p.ld = ld; p.N = N; p.M = M; p.Npad = round_up(N, 2); p.Nr = round_up(N, 128);
    p.eps = eps; p.max_iter = max_iter;
    p.demote = options().l2_demote != 1;
    const L2Plan l2 = l2_plan(8.0 * (double)ld * M, plan.grid, 8.0 * (double)ld * plan.A, ((M + plan.grid - 1) / plan.grid + plan.A - 1) / plan.A, plan.dynamic);
    p.resident_groups = l2.resident_groups; p.pingpong = l2.pingpong; p.pin_margin = l2.pin_margin;
    if (plan.A == 16) return launch_f64<16, 1>(p, plan, di.device, s);
    if (plan.A == 8) return launch_f64<8, 2>(p, plan, di.device, s);
    if (plan.A == 4) return launch_f64<4, 4>(p, plan, di.device, s);
    if (plan.dynamic) return launch_f64<2, 8, true>(p, plan, di.device, s);
    return launch_f64<2, 8>(p, plan, di.device, s);
}

}  // extern "C"
