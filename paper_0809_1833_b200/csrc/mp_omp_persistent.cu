// mp_omp_persistent.cu -- Orthogonal MP as ONE persistent cooperative kernel (omp_algo 1; mp_omp.cu is the stream loop).
//
// Selection: the register-streaming correlate + packed argmax of mp_persistent_ldg.cu (Eq. 9 / Eq. 16), unchanged, one
// item per warp in flight across the barriers.  Refit: the same float64 QR as the stream loop (Gram-Schmidt twice), but
// DISTRIBUTED BY COMPONENTS: CTA b owns the slice [b N/G, (b+1) N/G) of every basis vector and keeps it in shared memory
// for the whole solve (t x N/G doubles, 57 KB at t = 256, N = 4096), so the basis never travels.  Per iteration:
//     barrier 1   winning key (as MP)
//     partial h = Q_slice^T psi_i,slice -> global [cta][j]            barrier 2
//     CTA j mod G adds the G partials of h_j in a fixed order           barrier 3
//     w_slice = psi_i,slice - Q_slice h ; partial ||w||^2, <w, r> and the slice of w -> global           barrier 4
//     (a second Gram-Schmidt pass, three more barriers, only if ||w||^2 < ||psi_i||^2 / 2: the usual criterion)
//     everybody: ||w||^2, <w, r> (fixed order), r <- r - (<w,r>/||w||^2) w on its own full copy of r, ||r||^2, stop test;
//     q_t,slice = w_slice / ||w|| joins the CTA's basis slice.
// R, z and the selected atoms go to the workspace; x~ is produced by the stream loop's back-substitution kernel.
#include "mp_common.cuh"
#include "mp_internal.h"
#include "mp_omp.h"

namespace mp {

constexpr int kOmpPMaxWarps = 32;
constexpr int kOmpJGroups = 16;

struct OmpPParams {
    const float* psi_t;
    const float* y;
    int* idx_trace;
    OmpWs ws;
    int64_t ld;
    int N, M, Npad, Nr, T, Tld;
    int SLp;                    // padded (odd) pitch of a basis-vector slice in shared memory
    int atoms_max;
    float eps;
    int demote;                 // hand the pinned rows back at the end (knob l2_demote, default on)
    int resident_groups;        // groups of A atoms per CTA loaded L2::evict_last (mp_common.cuh), 0 = no hints
    int pingpong, pin_margin;   // DYN kernels: reversed item order on odd iterations, unpinned groups at either end (mp_internal.h l2_plan)
};

__device__ __forceinline__ float4 omp_ldg_cg4(const float4* p)
{
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// DYN (long shares, the HBM-streaming regime): warps draw their work items from a shared-memory counter, as in mp_persistent_ldg.cu
template <int A, int UC, bool DYN>
__global__ void __launch_bounds__(512, 1)
mp_omp_persistent_kernel(const OmpPParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int THREADS = blockDim.x, W = THREADS >> 5;
    const int G = gridDim.x, b = blockIdx.x;
    const OmpWs& ws = p.ws;

    double* r64 = reinterpret_cast<double*>(smem_raw);                         // Nr   residual, replicated in every CTA
    float* r32 = reinterpret_cast<float*>(r64 + p.Nr);                         // Nr   its fp32 rounding (feeds the dots)
    unsigned long long* wkey = reinterpret_cast<unsigned long long*>(r32 + p.Nr);
    double* red = reinterpret_cast<double*>(wkey + kOmpPMaxWarps);             // 32
    unsigned long long* skey = reinterpret_cast<unsigned long long*>(red + kOmpPMaxWarps);
    int* next_item = reinterpret_cast<int*>(skey + 1);                          // DYN: items beyond the first W are drawn from this counter
    double* wsl = reinterpret_cast<double*>(skey + 2);                         // SLp  slice of the direction being orthogonalised
    double* hbuf = wsl + p.SLp;                                                // Tld  reduced Q^T w of the current pass
    double* psum = hbuf + p.Tld;                                               // kOmpJGroups x SLp
    double* Qs = psum + kOmpJGroups * p.SLp;                                   // T x SLp  this CTA's slice of the basis
    float* part = reinterpret_cast<float*>(Qs + (size_t)p.T * p.SLp);          // [atom of this CTA][chunk]

    const int a0 = (int)(((int64_t)b * p.M) / G);
    const int a1 = (int)(((int64_t)(b + 1) * p.M) / G);
    const int n_atoms = a1 - a0;
    const int n_groups = (n_atoms + A - 1) / A;
    const int n4 = p.Npad >> 2;
    const int n_chunks = (n4 + 32 * UC - 1) / (32 * UC);
    const int n_items = n_groups * n_chunks;
    const bool ragged = p.Npad != p.N;
    const int s0 = (int)(((int64_t)b * p.N) / G), s1 = (int)(((int64_t)(b + 1) * p.N) / G);
    const int SL = s1 - s0;                                                    // components owned by this CTA
    const int NJG = min(kOmpJGroups, max(1, THREADS / max(SL, 1)));

    unsigned long long episode = 0;
    auto grid_sync = [&]() {
        episode += 1;
        __syncthreads();
        if (tid == 0) {
            red_add_release_u64(ws.ctrl, 1ull);
            const unsigned long long target = episode * (unsigned long long)G;
            while (ld_acquire_u64(ws.ctrl) < target) {}
        }
        __syncthreads();
    };

    // ---- r <- y, ||y|| ----------------------------------------------------------------------------------------------------
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
    const double thresh = (double)p.eps * sqrt(rr);
    __syncthreads();

    const float4* r4 = reinterpret_cast<const float4*>(r32);
    float4 v[A][UC];
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
            const int rel = g * A + a < n_atoms ? g * A + a : n_atoms - 1;
            const float4* row = reinterpret_cast<const float4*>(p.psi_t + (int64_t)(a0 + rel) * p.ld);
#pragma unroll
            for (int u = 0; u < UC; u++) {
                const int j = jb + 32 * u;
                v[a][u] = j < n4 ? omp_ldg_cg4(row + j) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
    };
    // partial dots of the basis slice with the direction slice: hpart[b][j] = sum_n Qs[j][n] wsl[n], j < t
    auto partial_h = [&](int t) {
        for (int j = tid; j < t; j += THREADS) {
            const double* q = Qs + (size_t)j * p.SLp;
            double s = 0.0;
            for (int n = 0; n < SL; n++) s += q[n] * wsl[n];
            ws.hpart[(size_t)b * p.Tld + j] = s;
        }
    };
    // h_j for j = b, b + G, ... : the G partials added lane-strided then by an xor butterfly (fixed order)
    auto reduce_h = [&](int t) {
        for (int k = warp; b + k * G < t; k += W) {
            const int j = b + k * G;
            double s = 0.0;
            for (int c = lane; c < G; c += 32) s += __ldcg(ws.hpart + (size_t)c * p.Tld + j);
            s = warp_sum(s);
            if (lane == 0) ws.h[j] = s;
        }
    };
    // wsl -= Q_slice h  (h gathered into shared memory first); CTA 0 records h into column t of R
    auto subtract_projection = [&](int t, bool first) {
        for (int j = tid; j < t; j += THREADS) {
            const double hj = __ldcg(ws.h + j);
            hbuf[j] = hj;
            if (b == 0) {
                if (first) ws.Rm[(size_t)j * p.Tld + t] = hj; else ws.Rm[(size_t)j * p.Tld + t] += hj;
            }
        }
        __syncthreads();
        if (tid < SL * NJG) {
            const int n = tid % SL, jg = tid / SL;
            double s = 0.0;
            for (int j = jg; j < t; j += NJG) s += hbuf[j] * Qs[(size_t)j * p.SLp + n];
            psum[jg * p.SLp + n] = s;
        }
        __syncthreads();
        if (tid < SL) {
            double s = 0.0;
            for (int jg = 0; jg < NJG; jg++) s += psum[jg * p.SLp + tid];
            wsl[tid] -= s;
        }
        __syncthreads();
    };

    int it = warp;
    bool have = it < n_items;
    if (have) load_item(it, false);
    if (DYN && tid == 0) *next_item = W;
    __syncthreads();
    int t = 0;
    // ---- the loop: while ||r|| > eps ||y|| and t < T (the stop rule of MP) ------------------------------------------
    while ((sqrt(rr) > thresh) && (t < p.T)) {
        // ---------- Eq. 9: items dealt round-robin to the warps (DYN: drawn from a counter), one always in flight --------------
        while (have) {
            int nxt = it + W;
            if (DYN && lane == 0) nxt = atomicAdd(next_item, 1);
            const bool flip = DYN && p.pingpong && (t & 1);                    // odd iterations visit the items in reverse order (mp_persistent_ldg.cu)
            const int itm = flip ? n_items - 1 - it : it;
            const int g = itm / n_chunks, ch = itm - g * n_chunks;
            const int atom0 = g * A;
            const int jb = ch * 32 * UC + lane;
            float acc[A];
#pragma unroll
            for (int a = 0; a < A; a++) acc[a] = 0.f;
#pragma unroll
            for (int u = 0; u < UC; u++) {
                const int j = jb + 32 * u;
                float4 rv = j < n4 ? r4[j] : make_float4(0.f, 0.f, 0.f, 0.f);
                if (ragged && j == n4 - 1) {
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
        it = warp;
        have = it < n_items;
        if (have) load_item(it, DYN && p.pingpong && ((t + 1) & 1));           // next iteration's first item, ahead of the barriers
        __syncthreads();
        if (DYN && tid == 0) *next_item = W;                                   // nobody draws again before the next barriers
        unsigned long long best = 0ull;
        for (int a = tid; a < n_atoms; a += THREADS) {
            float c = part[a * n_chunks];
            for (int ch = 1; ch < n_chunks; ch++) c += part[a * n_chunks + ch];
            const unsigned long long k = pack_key(c, a0 + a);
            best = k > best ? k : best;
        }
        best = warp_max(best);
        if (lane == 0) wkey[warp] = best;
        __syncthreads();
        unsigned long long* slot_key = ws.ctrl + 1 + (t % 3);
        if (warp == 0) {
            unsigned long long k = lane < W ? wkey[lane] : 0ull;
            k = warp_max(k);
            if (lane == 0 && k) red_max_u64(slot_key, k);
        }
        grid_sync();                                                           // barrier 1: the winning key
        if (tid == 0) *skey = ld_relaxed_u64(slot_key);
        __syncthreads();
        const int i = key_index(*skey);

        // ---------- refit: w <- psi_i - Q Q^T psi_i -----------------------------------------------------------------------------
        const float* psi_i = p.psi_t + (int64_t)i * p.ld;
        if (tid < SL) wsl[tid] = (double)__ldg(psi_i + s0 + tid);
        __syncthreads();
        // Gram-Schmidt with the usual reorthogonalisation criterion: a second pass only if the first one removed more
        // than half of the atom's energy (||w||^2 < ||psi_i||^2 / 2); for incoherent atoms it almost never does.
        double nrm2 = 0.0, zn = 0.0;
        for (int pass = 0; pass < 2; pass++) {
            double pa = 0.0;
            if (pass == 0 && warp == 0) {
                for (int n = lane; n < SL; n += 32) pa += wsl[n] * wsl[n];
                pa = warp_sum(pa);
            }
            if (t > 0) {
                partial_h(t);
                grid_sync();                                                   // partial dots out
                reduce_h(t);
                grid_sync();                                                   // h reduced
                subtract_projection(t, pass == 0);
            }
            // ---------- ||w||^2, <w, r>, (||psi_i||^2) and the slice of w for everybody ------------------------------------
            if (warp == 0) {
                double pw = 0.0, pz = 0.0;
                for (int n = lane; n < SL; n += 32) { pw += wsl[n] * wsl[n]; pz += wsl[n] * r64[s0 + n]; }
                pw = warp_sum(pw);
                pz = warp_sum(pz);
                if (lane == 0) {
                    ws.scal[4 * b] = pw; ws.scal[4 * b + 1] = pz;
                    if (pass == 0) ws.scal[4 * b + 2] = pa;
                }
            }
            if (tid < SL) ws.w[s0 + tid] = wsl[tid];
            if (b == 0 && tid == 0 && pass == 0) st_relaxed_u64(ws.ctrl + 1 + ((t + 2) % 3), 0ull);   // key slot of t-1, reused at t+2
            grid_sync();                                                       // exchange
            if (warp == 0) {
                double nw = 0.0, z1 = 0.0, aa = 0.0;
                for (int c = lane; c < G; c += 32) {
                    nw += __ldcg(ws.scal + 4 * c); z1 += __ldcg(ws.scal + 4 * c + 1); aa += __ldcg(ws.scal + 4 * c + 2);
                }
                nw = warp_sum(nw);
                z1 = warp_sum(z1);
                aa = warp_sum(aa);
                if (lane == 0) { red[0] = nw; red[1] = z1; red[2] = aa; }
            }
            __syncthreads();
            nrm2 = red[0]; zn = red[1];
            const bool again = pass == 0 && t > 0 && nrm2 < 0.5 * red[2];
            __syncthreads();
            if (!again) break;
        }
        if (!(nrm2 > 1e-20)) break;                                            // the atom lies in the span of the selected ones
        const double nrm = sqrt(nrm2), coef = zn / nrm2;
        if (tid < SL) Qs[(size_t)t * p.SLp + tid] = wsl[tid] / nrm;            // q_t joins the basis slice
        double s2 = 0.0;
        for (int n = tid; n < p.N; n += THREADS) {                             // r <- r - <q_t, r> q_t on this CTA's full copy
            const double vn = r64[n] - coef * __ldcg(ws.w + n);
            r64[n] = vn;
            r32[n] = (float)vn;
            s2 += vn * vn;
        }
        s2 = warp_sum(s2);
        __syncthreads();
        if (lane == 0) red[warp] = s2;
        if (b == 0 && tid == 0) {
            ws.Rm[(size_t)t * p.Tld + t] = nrm;
            ws.z[t] = zn / nrm;
            ws.sel[t] = i;
            if (p.idx_trace) p.idx_trace[t] = i;
        }
        __syncthreads();
        rr = 0.0;
        for (int w = 0; w < W; w++) rr += red[w];
        __syncthreads();
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
    // ---- the state the back-substitution kernel needs: r (float64) and t ----------------------------------------------------------
    if (b == 0) {
        for (int n = tid; n < p.N; n += THREADS) ws.r64[n] = r64[n];
        if (tid == 0) ws.ctrl[kCtrT] = (unsigned long long)t;
    }
}

// ------------------------------------------------------------------------------------------------------------------
struct OmpPPlan {
    int A, UC, W, grid, SLp, atoms_max;
    size_t smem;
    bool dynamic;
};

static bool omp_p_plan(int N, int M, int T, const DeviceInfo& di, OmpPPlan* plan)
{
    if (!di.coop || di.sm_count < 1 || di.sm_count > kOmpMaxCtas || T < 1) return false;
    const int G = di.sm_count;
    const int n4 = round_up(N, 4) / 4;
    int A = 2, UC = 8;
    if (n4 <= 32) { A = 16; UC = 1; }
    else if (n4 <= 64) { A = 8; UC = 2; }
    else if (n4 <= 128) { A = 4; UC = 4; }
    const int atoms_max = (M + G - 1) / G;
    const int n_chunks = (n4 + 32 * UC - 1) / (32 * UC);
    const int items = ((atoms_max + A - 1) / A) * n_chunks;
    const int SL = (N + G - 1) / G;
    if (SL > 512) return false;
    const int SLp = SL | 1;
    const size_t Nr = (size_t)round_up(N, 128), Tld = (size_t)round_up(T, 32);
    const size_t smem = Nr * 12 + 8 * (2 * kOmpPMaxWarps + 2) + 8 * ((size_t)SLp + Tld + (size_t)kOmpJGroups * SLp + (size_t)T * SLp) +
                        4 * (size_t)atoms_max * n_chunks + 64;
    if (smem > (size_t)di.smem_optin) return false;
    int W = 16;
    double best = -1.0;
    for (int w = 8; w <= 16; w++) {
        const double fill = (double)items / ((double)((items + w - 1) / w) * w);
        if (fill >= best) { best = fill; W = w; }
    }
    plan->dynamic = A == 2 && items >= 8 * 16 && options().balance != 1;         // long shares: see mp_persistent_ldg.cu
    if (plan->dynamic) W = 16;
    if (W * 32 < SL) W = (SL + 31) / 32;
    plan->A = A; plan->UC = UC; plan->W = W; plan->grid = G; plan->SLp = SLp; plan->atoms_max = atoms_max; plan->smem = smem;
    return true;
}

bool omp_persistent_supported(int N, int M, int T)
{
    DeviceInfo di;
    if (device_info(&di) != MP_OK) return false;
    OmpPPlan plan;
    return omp_p_plan(N, M, T, di, &plan);
}

template <int A, int UC, bool DYN = false>
static mp_status launch_omp_p(const OmpPParams& p, const OmpPPlan& plan, int device, cudaStream_t stream)
{
    static thread_local int attr_dev = -1;
    if (attr_dev != device) {
        MP_CUDA(cudaFuncSetAttribute(mp_omp_persistent_kernel<A, UC, DYN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        attr_dev = device;
    }
    int occ = 0;
    MP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mp_omp_persistent_kernel<A, UC, DYN>, plan.W * 32, plan.smem));
    if (occ < 1) return fail(MP_ERR_UNSUPPORTED, "persistent Orthogonal MP kernel does not fit one CTA per SM");
    void* args[] = {(void*)&p};
    MP_CUDA(cudaLaunchCooperativeKernel((const void*)mp_omp_persistent_kernel<A, UC, DYN>, dim3(plan.grid), dim3(plan.W * 32), args,
                                        plan.smem, stream));
    count_launch();
    return MP_OK;
}

mp_status launch_omp_persistent(const OmpArgs& a, const OmpWs& ws, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    OmpPPlan plan;
    if (!omp_p_plan(a.N, a.M, a.T, di, &plan))
        return fail(MP_ERR_UNSUPPORTED, "N=%d, M=%d, T=%d do not fit the persistent Orthogonal MP kernel's shared memory", a.N, a.M, a.T);
    MP_CUDA(cudaMemsetAsync(ws.ctrl, 0, 256, stream));
    OmpPParams p;
    p.psi_t = a.psi_t; p.y = a.y; p.idx_trace = a.idx_trace; p.ws = ws; p.ld = a.ld;
    p.N = a.N; p.M = a.M; p.Npad = round_up(a.N, 4); p.Nr = round_up(a.N, 128); p.T = a.T; p.Tld = round_up(a.T, 32);
    p.SLp = plan.SLp; p.atoms_max = plan.atoms_max; p.eps = a.eps;
    p.demote = options().l2_demote != 1;
    const L2Plan l2 = l2_plan(4.0 * (double)a.ld * a.M, plan.grid, 4.0 * (double)a.ld * plan.A, ((a.M + plan.grid - 1) / plan.grid + plan.A - 1) / plan.A, plan.dynamic);
    p.resident_groups = l2.resident_groups; p.pingpong = l2.pingpong; p.pin_margin = l2.pin_margin;
    if (plan.A == 16) return launch_omp_p<16, 1>(p, plan, di.device, stream);
    if (plan.A == 8) return launch_omp_p<8, 2>(p, plan, di.device, stream);
    if (plan.A == 4) return launch_omp_p<4, 4>(p, plan, di.device, stream);
    if (plan.dynamic) return launch_omp_p<2, 8, true>(p, plan, di.device, stream);
    return launch_omp_p<2, 8>(p, plan, di.device, stream);
}

}  // namespace mp
