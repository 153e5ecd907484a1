// mp_persistent.cu -- "algo 1": the whole MP loop (Eq. 8-12) as ONE persistent cooperative kernel.
//
// Design (DESIGN.md section "Persistent kernel"):
//   * grid = one CTA per SM, co-resident (cooperative launch); CTA b owns the contiguous atom range
//     [b*M/G, (b+1)*M/G) of the atom-major dictionary, balanced to one atom.
//   * every warp owns D private shared-memory stages ("slots") and streams its share of the CTA's atoms
//     through them with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx); the warp refills a
//     slot itself right after consuming it, so there is no producer warp and no cross-warp handshake.
//     Psi never changes, so the refill for the NEXT iteration is issued before the grid barrier:
//     the HBM stream does not stop at the iteration boundary.
//   * correlations (Eq. 9) are fp32 dot products against an fp32 copy of r in shared memory; each warp
//     carries a packed (|c|, index, sign) key (Eq. 16, lowest index on ties); block max -> one
//     red.max.u64 per CTA -> ONE grid barrier per iteration (monotonic counter, release/acquire).
//   * after the barrier every CTA applies r <- r - c psi_i (Eq. 11) to its OWN float64 copy of r in
//     shared memory (psi_i is 4N bytes from L2) and recomputes ||r||^2 as a direct float64 sum (Eq. 18)
//     in a fixed order, so all CTAs take the same stop decision without a second barrier.
//   * CTA 0 additionally does x~_i += c (Eq. 10, float64 accumulators in the workspace) and the traces.
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kMaxWarps = 24;
constexpr int kMaxThreads = kMaxWarps * 32;
constexpr int kMaxAtomsPerItem = 32;

struct PersistentParams {
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
    int N, M, Npad, Nr;         // Npad = N rounded up to 4, Nr = N rounded up to 128
    int A;                      // atoms per item (KC == 1), else 1
    int KC;                     // column chunks per atom
    int BN;                     // columns per chunk (multiple of 128) when KC > 1; Npad when KC == 1
    int D;                      // slots per warp
    int slot_floats;
    int contiguous;             // 1 if ld == Npad (an item's atoms are one contiguous byte range)
    float eps;
    int max_iter;
};

// lane-strided fp32 dot product of one shared-memory row with the fp32 residual (cols % 4 == 0)
__device__ __forceinline__ float dot_row(const float* __restrict__ row, const float* __restrict__ rv, int cols, int lane)
{
    const float4* p4 = reinterpret_cast<const float4*>(row);
    const float4* r4 = reinterpret_cast<const float4*>(rv);
    const int n4 = cols >> 2;
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
    int j = lane;
    for (; j + 96 < n4; j += 128) {
        const float4 a = p4[j], b = p4[j + 32], c = p4[j + 64], d = p4[j + 96];
        const float4 u = r4[j], v = r4[j + 32], w = r4[j + 64], z = r4[j + 96];
        s0 = fmaf(a.x, u.x, s0); s0 = fmaf(a.y, u.y, s0); s0 = fmaf(a.z, u.z, s0); s0 = fmaf(a.w, u.w, s0);
        s1 = fmaf(b.x, v.x, s1); s1 = fmaf(b.y, v.y, s1); s1 = fmaf(b.z, v.z, s1); s1 = fmaf(b.w, v.w, s1);
        s2 = fmaf(c.x, w.x, s2); s2 = fmaf(c.y, w.y, s2); s2 = fmaf(c.z, w.z, s2); s2 = fmaf(c.w, w.w, s2);
        s3 = fmaf(d.x, z.x, s3); s3 = fmaf(d.y, z.y, s3); s3 = fmaf(d.z, z.z, s3); s3 = fmaf(d.w, z.w, s3);
    }
    for (; j < n4; j += 32) {
        const float4 a = p4[j];
        const float4 u = r4[j];
        s0 = fmaf(a.x, u.x, s0); s0 = fmaf(a.y, u.y, s0); s0 = fmaf(a.z, u.z, s0); s0 = fmaf(a.w, u.w, s0);
    }
    return (s0 + s1) + (s2 + s3);
}

// two rows at once, sharing the residual loads
__device__ __forceinline__ void dot_row2(const float* __restrict__ row0, const float* __restrict__ row1,
                                         const float* __restrict__ rv, int cols, int lane, float& o0, float& o1)
{
    const float4* p4 = reinterpret_cast<const float4*>(row0);
    const float4* q4 = reinterpret_cast<const float4*>(row1);
    const float4* r4 = reinterpret_cast<const float4*>(rv);
    const int n4 = cols >> 2;
    float s0 = 0.f, s1 = 0.f, t0 = 0.f, t1 = 0.f;
    int j = lane;
    for (; j + 32 < n4; j += 64) {
        const float4 a = p4[j], b = p4[j + 32], c = q4[j], d = q4[j + 32];
        const float4 u = r4[j], v = r4[j + 32];
        s0 = fmaf(a.x, u.x, s0); s0 = fmaf(a.y, u.y, s0); s0 = fmaf(a.z, u.z, s0); s0 = fmaf(a.w, u.w, s0);
        s1 = fmaf(b.x, v.x, s1); s1 = fmaf(b.y, v.y, s1); s1 = fmaf(b.z, v.z, s1); s1 = fmaf(b.w, v.w, s1);
        t0 = fmaf(c.x, u.x, t0); t0 = fmaf(c.y, u.y, t0); t0 = fmaf(c.z, u.z, t0); t0 = fmaf(c.w, u.w, t0);
        t1 = fmaf(d.x, v.x, t1); t1 = fmaf(d.y, v.y, t1); t1 = fmaf(d.z, v.z, t1); t1 = fmaf(d.w, v.w, t1);
    }
    for (; j < n4; j += 32) {
        const float4 a = p4[j], c = q4[j];
        const float4 u = r4[j];
        s0 = fmaf(a.x, u.x, s0); s0 = fmaf(a.y, u.y, s0); s0 = fmaf(a.z, u.z, s0); s0 = fmaf(a.w, u.w, s0);
        t0 = fmaf(c.x, u.x, t0); t0 = fmaf(c.y, u.y, t0); t0 = fmaf(c.z, u.z, t0); t0 = fmaf(c.w, u.w, t0);
    }
    o0 = s0 + s1;
    o1 = t0 + t1;
}

__global__ void __launch_bounds__(kMaxThreads, 1)
mp_persistent_kernel(const PersistentParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int W = blockDim.x >> 5, nthreads = blockDim.x;
    const int G = gridDim.x;

    // ---- shared memory carve-up ------------------------------------------------------------------------
    double* r64 = reinterpret_cast<double*>(smem_raw);                         // Nr doubles (master residual)
    float* r32 = reinterpret_cast<float*>(r64 + p.Nr);                         // Nr floats  (fp32 rounding, feeds the dots)
    float* slots = r32 + p.Nr;                                                 // W*D*slot_floats (16-B aligned: Nr % 128 == 0)
    uint64_t* full = reinterpret_cast<uint64_t*>(slots + (size_t)W * p.D * p.slot_floats);   // W*D mbarriers
    unsigned long long* wkey = reinterpret_cast<unsigned long long*>(full + W * p.D);        // W
    double* red = reinterpret_cast<double*>(wkey + kMaxWarps);                 // W
    unsigned long long* skey = reinterpret_cast<unsigned long long*>(red + kMaxWarps);       // 1

    // ---- this CTA's atoms, this warp's items --------------------------------------------------------------
    const int a0 = (int)(((int64_t)blockIdx.x * p.M) / G);
    const int a1 = (int)(((int64_t)(blockIdx.x + 1) * p.M) / G);
    const int n_groups = (a1 - a0 + p.A - 1) / p.A;                            // groups of A consecutive atoms
    const int ng_w = warp < n_groups ? (n_groups - warp + W - 1) / W : 0;      // groups warp, warp+W, ...
    const int n_items = ng_w * p.KC;                                           // items per iteration of this warp
    const bool stationary = n_items <= p.D;                                    // whole share fits: load once, never refill
    float* my_slots = slots + (size_t)warp * p.D * p.slot_floats;
    uint64_t* my_full = full + warp * p.D;

    if (lane == 0)
        for (int d = 0; d < p.D; d++) mbar_init(my_full + d, 1);
    mbar_fence_init();
    __syncthreads();

    // issue the TMA copies of item `il` (index within one iteration) into slot `slot`
    auto issue_item = [&](int il, int slot) {
        const int gl = il / p.KC, k = il - gl * p.KC;
        const int atom0 = a0 + (warp + gl * W) * p.A;
        const int na = min(p.A, a1 - atom0);
        const int col0 = k * p.BN;
        const int cc = min(p.BN, p.Npad - col0);
        float* dst = my_slots + (size_t)slot * p.slot_floats;
        uint64_t* bar = my_full + slot;
        fence_proxy_async_smem();                                              // our earlier generic accesses to the slot
        if (lane == 0) mbar_arrive_expect_tx(bar, (uint32_t)(na * cc * 4));
        __syncwarp();
        if (p.contiguous && p.KC == 1) {
            if (lane == 0) tma_load_1d(dst, p.psi_t + (int64_t)atom0 * p.ld, (uint32_t)(na * cc * 4), bar);
        } else if (lane < na) {
            tma_load_1d(dst + (size_t)lane * cc, p.psi_t + (int64_t)(atom0 + lane) * p.ld + col0, (uint32_t)(cc * 4), bar);
        }
    };

    int issued = 0, consumed = 0;                                               // running item counts of this warp
    {
        const int first = min(n_items, p.D);
        for (; issued < first; issued++) issue_item(issued, issued);
    }

    // ---- Eq. 8: r <- y (float64 master + fp32 copy), ||y||^2 ------------------------------------------------
    double ss = 0.0;
    for (int n = tid; n < p.Nr; n += nthreads) {
        const float v = n < p.N ? p.y[n] : 0.f;
        r64[n] = (double)v;
        r32[n] = v;
        ss += (double)v * (double)v;
    }
    ss = warp_sum(ss);
    if (lane == 0) red[warp] = ss;
    __syncthreads();
    double rr = warp_sum(lane < W ? red[lane] : 0.0);
    const double yy = rr;
    const double thresh = (double)p.eps * sqrt(yy);
    __syncthreads();

    int t = 0;
    float acc = 0.f;                                                            // per-lane partial of a chunked atom (KC > 1)
    // ---- the loop: while ||r|| > eps ||y|| and t < T ----------------------------------------------------
    while ((sqrt(rr) > thresh) && (t < p.max_iter)) {
        // ---------- Eq. 9 + Eq. 16: stream this warp's atoms, fp32 dots, running packed argmax ---------------
        unsigned long long best = 0ull;
        for (int il = 0; il < n_items; il++) {
            int slot;
            if (stationary) {
                slot = il;
                if (t == 0) { mbar_wait(my_full + slot, 0); consumed++; }
            } else {
                slot = consumed % p.D;
                mbar_wait(my_full + slot, (uint32_t)((consumed / p.D) & 1));
                consumed++;
            }
            const int gl = il / p.KC, k = il - gl * p.KC;
            const int atom0 = a0 + (warp + gl * W) * p.A;
            const int na = min(p.A, a1 - atom0);
            const int col0 = k * p.BN;
            const int cc = min(p.BN, p.Npad - col0);
            float* s = my_slots + (size_t)slot * p.slot_floats;
            if (p.Npad != p.N && col0 + cc == p.Npad && (!stationary || t == 0)) {
                // N % 4 != 0: the copies brought up to 3 caller-owned pad floats per atom; zero them
                if (lane < na)
                    for (int c = p.N - col0; c < cc; c++) s[(size_t)lane * cc + c] = 0.f;
                __syncwarp();
            }
            if (p.KC == 1) {
                int j = 0;
                for (; j + 1 < na; j += 2) {
                    float c0, c1;
                    dot_row2(s + (size_t)j * cc, s + (size_t)(j + 1) * cc, r32, cc, lane, c0, c1);
                    c0 = warp_sum(c0);
                    c1 = warp_sum(c1);
                    const unsigned long long k0 = pack_key(c0, atom0 + j), k1 = pack_key(c1, atom0 + j + 1);
                    best = k0 > best ? k0 : best;
                    best = k1 > best ? k1 : best;
                }
                if (j < na) {
                    const float c0 = warp_sum(dot_row(s + (size_t)j * cc, r32, cc, lane));
                    const unsigned long long k0 = pack_key(c0, atom0 + j);
                    best = k0 > best ? k0 : best;
                }
            } else {
                acc += dot_row(s, r32 + col0, cc, lane);
                if (k == p.KC - 1) {
                    const float c0 = warp_sum(acc);
                    acc = 0.f;
                    const unsigned long long k0 = pack_key(c0, atom0);
                    best = k0 > best ? k0 : best;
                }
            }
            // refill this slot with the item D positions ahead in the cyclic item sequence (possibly next iteration's)
            if (!stationary) {
                const int ahead = il + p.D;
                const int t_ahead = t + ahead / n_items;
                if (t_ahead < p.max_iter) {
                    __syncwarp();
                    issue_item(ahead % n_items, slot);
                    issued++;
                }
            }
        }

        // ---------- block argmax -> grid argmax, ONE grid barrier (mp_common.cuh) ---------------------------------------------
        const unsigned long long key = grid_argmax(best, wkey, skey, p.ctrl, t);
        const int i = key_index(key);
        const float c = key_value(key);
        const double cd = (double)c;

        // ---------- Eq. 11 on this CTA's float64 r, Eq. 18 direct sum ------------------------------------------------
        {
            const float4* psi4 = reinterpret_cast<const float4*>(p.psi_t + (int64_t)i * p.ld);
            double s2 = 0.0;
            for (int j = tid; j < (p.Npad >> 2); j += nthreads) {
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
            s2 = warp_sum(s2);
            if (lane == 0) red[warp] = s2;
        }
        // ---------- Eq. 10, Eq. 12, traces: CTA 0 only ---------------------------------------------------------------
        if (blockIdx.x == 0 && tid == 0) {
            record_step(p.x64, p.idx_trace, p.c_trace, p.ctrl, t, i, c);
        }
        __syncthreads();
        rr = warp_sum(lane < W ? red[lane] : 0.0);
        t += 1;
    }

    // ---- drain prefetches that will never be consumed -----------------------------------------------------------------
    if (!stationary) {
        while (consumed < issued) {
            mbar_wait(my_full + (consumed % p.D), (uint32_t)((consumed / p.D) & 1));
            consumed++;
        }
    } else if (t == 0) {
        for (int d = 0; d < issued; d++) mbar_wait(my_full + d, 0);
    }

    // ---- P:86 return x~ (and r, t): CTA 0 -------------------------------------------------------------------------------
    if (blockIdx.x == 0) {
        if (tid == 0) __threadfence();
        __syncthreads();
        for (int m = tid; m < p.M; m += nthreads) p.x[m] = (float)__ldcg(p.x64 + m);
        for (int n = tid; n < p.N; n += nthreads) p.r[n] = r32[n];
        if (tid == 0) *p.n_iter = t;
    }
}

// ------------------------------------------------------------------------------------------------------------------
struct PersistentPlan {
    int W, D, A, KC, BN, slot_floats, grid;
    size_t smem;
};

static bool make_plan(int N, int M, const DeviceInfo& di, PersistentPlan* plan)
{
    const Options& o = options();
    const int Npad = round_up(N, 4), Nr = round_up(N, 128);
    const size_t fixed = (size_t)Nr * 12 + 8 * (2 * kMaxWarps + 2) + 128;
    if (fixed + 4 * 4096 > (size_t)di.smem_optin) return false;
    const size_t avail = (size_t)di.smem_optin - fixed;
    const int row_bytes = Npad * 4;
    int target_slot = o.slot_bytes > 0 ? (int)o.slot_bytes : 8192;
    int A = 1, KC = 1, BN = Npad, slot_bytes;
    if (row_bytes <= target_slot) {
        A = target_slot / row_bytes;
        if (A > kMaxAtomsPerItem) A = kMaxAtomsPerItem;
        slot_bytes = A * row_bytes;
    } else {
        KC = (row_bytes + target_slot - 1) / target_slot;
        BN = round_up((Npad + KC - 1) / KC, 128);
        KC = (Npad + BN - 1) / BN;
        slot_bytes = BN * 4;
    }
    int W, D;
    const int max_slots = (int)((avail - 8 * 0) / (slot_bytes + 8));
    if (max_slots < 1) return false;
    if (o.warps > 0) {
        W = (int)o.warps;
        if (W > kMaxWarps) W = kMaxWarps;
        D = o.depth > 0 ? (int)o.depth : max_slots / W;
    } else if (o.depth > 0) {
        D = (int)o.depth;
        W = max_slots / D;
    } else {
        // Choose the warp count for BALANCE.  The CTA with the most atoms sets the iteration time, and a warp works
        // through its groups one after another, so what counts is rounds = ceil(groups / W): with 111 atoms, 22 warps
        // need 6 rounds of which the last is 16 % full (measured 47.9 us per iteration at CFG3), 16 warps need 7 full
        // rounds (43.6 us).  Score = fill of the rounds, scaled down if fewer than 96 KB can be in flight (HBM latency x
        // per-SM bandwidth share is about 88 KB); a share that fits entirely in the slots (stationary dictionary)
        // beats everything.  Ties go to more warps.
        const int G = di.sm_count > 0 ? di.sm_count : 1;
        const int atoms_max = (M + G - 1) / G;
        const int groups = (atoms_max + A - 1) / A;
        double best_score = -1.0;
        W = 1; D = 1;
        for (int w = 1; w <= kMaxWarps; w++) {
            int d = max_slots / w;
            if (d < 1) break;
            if (w < 8 && max_slots >= 8 && groups > w) continue;              // fewer than 8 warps cannot keep up with the stream
            if (d > 64) d = 64;
            const int per_warp_items = ((groups + w - 1) / w) * KC;
            const bool fits = per_warp_items <= d;
            const double fill = (double)groups / ((double)((groups + w - 1) / w) * w);
            const double inflight = (double)w * (double)(d < per_warp_items ? d : per_warp_items) * slot_bytes;
            double score = fill * (inflight >= 96.0 * 1024 ? 1.0 : inflight / (96.0 * 1024));
            if (fits) score = 10.0 + fill;
            if (score >= best_score) { best_score = score; W = w; D = d; }
        }
    }
    if (W > kMaxWarps) W = kMaxWarps;
    if (W < 1 || D < 1) return false;
    if (D > 64) D = 64;
    if ((size_t)W * D * (slot_bytes + 8) > avail) return false;
    plan->W = W; plan->D = D; plan->A = A; plan->KC = KC; plan->BN = BN;
    plan->slot_floats = slot_bytes / 4;
    plan->grid = o.grid > 0 ? (int)o.grid : di.sm_count;
    if (plan->grid > di.sm_count) plan->grid = di.sm_count;
    plan->smem = fixed + (size_t)W * D * (slot_bytes + 8);
    return true;
}

bool persistent_supported(int N, int M)
{
    DeviceInfo di;
    if (device_info(&di) != MP_OK || !di.coop) return false;
    PersistentPlan plan;
    return make_plan(N, M, di, &plan);
}

mp_status launch_recover_persistent(const RecoverArgs& a, const Workspace& ws, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    if (!di.coop) return fail(MP_ERR_UNSUPPORTED, "device does not support cooperative launch");
    PersistentPlan plan;
    if (!make_plan(a.N, a.M, di, &plan))
        return fail(MP_ERR_UNSUPPORTED, "N=%d does not fit the persistent kernel's shared-memory plan", a.N);

    static thread_local int smem_set_for_device = -1;
    if (smem_set_for_device != di.device) {
        MP_CUDA(cudaFuncSetAttribute(mp_persistent_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, di.smem_optin));
        smem_set_for_device = di.device;
    }
    int occ = 0;
    MP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mp_persistent_kernel, plan.W * 32, plan.smem));
    if (occ < 1) return fail(MP_ERR_UNSUPPORTED, "persistent kernel does not fit one CTA per SM (smem %zu)", plan.smem);

    // control block and the float64 coefficient accumulators start at zero (Eq. 8)
    MP_CUDA(cudaMemsetAsync(ws.ctrl, 0, 256 + sizeof(double) * (size_t)a.M, stream));

    PersistentParams p;
    p.psi_t = a.psi_t; p.y = a.y; p.x = a.x; p.r = a.r; p.n_iter = a.n_iter;
    p.idx_trace = a.idx_trace; p.c_trace = a.c_trace;
    p.x64 = ws.x64; p.ctrl = ws.ctrl; p.ld = a.ld;
    p.N = a.N; p.M = a.M; p.Npad = round_up(a.N, 4); p.Nr = round_up(a.N, 128);
    p.A = plan.A; p.KC = plan.KC; p.BN = plan.BN; p.D = plan.D; p.slot_floats = plan.slot_floats;
    p.contiguous = (a.ld == p.Npad) ? 1 : 0;
    p.eps = a.eps; p.max_iter = a.max_iter;
    void* args[] = {(void*)&p};
    MP_CUDA(cudaLaunchCooperativeKernel((const void*)mp_persistent_kernel, dim3(plan.grid), dim3(plan.W * 32), args,
                                        plan.smem, stream));
    count_launch();
    return MP_OK;
}

}  // namespace mp
