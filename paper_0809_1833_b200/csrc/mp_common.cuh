// mp_common.cuh -- shared device helpers of the B200 Matching Pursuit kernels (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mp {

// ------------------------------------------------------------------------------------------------
// Packed argmax key (Eq. 9 / Eq. 16: largest |c|, smallest index on ties).
//   bits 63..32  float bits of |c|   (|c| >= 0, so IEEE bits order as unsigned ints; NaN -> 0)
//   bits 31..1   0x7FFFFFFF - index  (lower index = larger key)
//   bit  0       sign bit of c       (rides along so the signed c is recovered without a second read)
// max() over keys is exact and order-independent, so a block/grid reduction by atomicMax is deterministic.
// Every real key is > 0 (index < 0x7FFFFFFF), so 0 is the "empty" value of a key slot.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long pack_key(float c, int index)
{
    unsigned int bits = __float_as_uint(c);
    unsigned int mag = bits & 0x7FFFFFFFu;
    if (mag > 0x7F800000u) mag = 0u;                       // NaN never wins
    unsigned int lo = ((0x7FFFFFFFu - (unsigned int)index) << 1) | (bits >> 31);
    return ((unsigned long long)mag << 32) | lo;
}
__device__ __forceinline__ int key_index(unsigned long long key)
{
    return (int)(0x7FFFFFFFu - ((unsigned int)(key & 0xFFFFFFFFull) >> 1));
}
__device__ __forceinline__ float key_value(unsigned long long key)
{
    unsigned int mag = (unsigned int)(key >> 32);
    unsigned int sign = (unsigned int)(key & 1ull) << 31;
    return __uint_as_float(mag | sign);
}

// ------------------------------------------------------------------------------------------------
// Warp reductions.  xor-butterflies with a commutative op leave the bit-identical result in every lane.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// 64-bit max over the warp with two hardware reductions (REDUX): the high words first, then the low words of the lanes that hold
// the winning high word.  Same result as the butterfly below in a fifth of the latency.
__device__ __forceinline__ unsigned long long warp_max_redux(unsigned long long k)
{
    const unsigned int hi = (unsigned int)(k >> 32);
    const unsigned int m = __reduce_max_sync(0xffffffffu, hi);
    const unsigned int lo = __reduce_max_sync(0xffffffffu, hi == m ? (unsigned int)k : 0u);
    return ((unsigned long long)m << 32) | lo;
}
__device__ __forceinline__ unsigned long long warp_max(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = w > v ? w : v;
    }
    return v;
}

// ------------------------------------------------------------------------------------------------
// mbarrier + TMA bulk-copy PTX (sm_90+/sm_100a).  SASS: SYNCS.*, UBLKCP.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
// generic-proxy accesses to shared memory before this fence are ordered before later async-proxy (TMA) accesses
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// 1-D bulk copy global -> shared, completion reported on an mbarrier (bytes % 16 == 0, 16-B aligned both sides)
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ------------------------------------------------------------------------------------------------
// gpu-scope atomics / ordered accesses used by the grid barrier
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void red_max_u64(unsigned long long* p, unsigned long long v)
{
    asm volatile("red.relaxed.gpu.global.max.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void red_add_release_u64(unsigned long long* p, unsigned long long v)
{
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void red_add_f64(double* p, double v)
{
    asm volatile("red.relaxed.gpu.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// ------------------------------------------------------------------------------------------------
// The iteration boundary shared by the grid-wide fp32 kernels (mp_persistent_ldg.cu, mp_persistent.cu, mp_signs.cu):
// block argmax -> grid argmax with ONE grid barrier (Eq. 9 / Eq. 16), and CTA 0's bookkeeping of the step (Eq. 10, traces).
//   ctrl[0]     monotonic arrive counter (iteration t is complete at (t + 1) * gridDim.x)
//   ctrl[1..3]  key slots rotating with t mod 3: slot t is filled by red.max before the arrive, read after the spin, and
//               zeroed again by CTA 0 during iteration t + 1 (every CTA has read it by then), two iterations before its reuse
// All threads of every CTA call grid_argmax with their warp's best key; every thread gets the same winning key back.
// wkey: kMaxWarps shared slots, skey: one shared slot.  Four dependent L2 hops (max acknowledged by the release fence ->
// arrive -> spin -> key read); cheaper schemes were measured and lost at 148 CTAs (profiles/k1_boundary_r02.md).
// stamp_arrive / stamp_done (profiling builds): clock64 of thread 0 after the arrive and after the spin.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long grid_argmax(unsigned long long warp_best, unsigned long long* wkey, unsigned long long* skey,
                                                          unsigned long long* ctrl, int t, long long* stamp_arrive = nullptr,
                                                          long long* stamp_done = nullptr)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    if (lane == 0) wkey[warp] = warp_best;
    __syncthreads();
    if (warp == 0) {
        unsigned long long k = lane < W ? wkey[lane] : 0ull;
        k = warp_max_redux(k);
        if (lane == 0) {
            unsigned long long* slot_key = ctrl + 1 + (t % 3);
            if (k) red_max_u64(slot_key, k);
            red_add_release_u64(ctrl, 1ull);
            if (stamp_arrive) *stamp_arrive = clock64();
            const unsigned long long target = (unsigned long long)(t + 1) * (unsigned long long)gridDim.x;
            while (ld_acquire_u64(ctrl) < target) {}
            if (stamp_done) *stamp_done = clock64();
            *skey = ld_relaxed_u64(slot_key);
        }
    }
    __syncthreads();
    return *skey;
}
// one thread of CTA 0 (not the thread every CTA's barrier waits for): x~_i += c in float64 (Eq. 10), the traces, and the key slot
// of iteration t - 1 handed back
__device__ __forceinline__ void record_step(double* x64, int* idx_trace, float* c_trace, unsigned long long* ctrl, int t, int i, float c)
{
    red_add_f64(x64 + i, (double)c);
    if (idx_trace) idx_trace[t] = i;
    if (c_trace) c_trace[t] = c;
    st_relaxed_u64(ctrl + 1 + ((t + 2) % 3), 0ull);
}

// ------------------------------------------------------------------------------------------------
// L2 residency control.  A dictionary larger than L2, streamed cyclically, gets no reuse at all (ncu: DRAM traffic = 4NM
// per iteration, L2 hit rate 0.2 %).  Loading a FIXED subset of the rows with the evict_last priority and the rest with
// evict_first keeps that subset in L2 across iterations, so only the rest comes from HBM every iteration.  Measured on
// B200 (profiles/persistent_r01.md): ~64-72 MB stay resident (more thrashes), CFG3 40.5 -> 33.2 us per iteration.
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ float4 ldg_cg4_hint(const float4* p, uint64_t policy)
{
    float4 v;
    asm volatile("ld.global.cg.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(policy));
    return v;
}

__device__ __forceinline__ double2 ldg_cg_d2_hint(const double2* p, uint64_t policy)
{
    double2 v;
    asm volatile("ld.global.cg.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(policy));
    return v;
}
// group g of n_groups is one of the rg resident ones (spread evenly: L2 hits and HBM misses interleave in time)
__device__ __forceinline__ bool l2_group_is_resident(int g, int rg, int n_groups)
{
    return ((long long)(g + 1) * rg) / n_groups != ((long long)g * rg) / n_groups;
}

// At the end of a solve the rows that were pinned with evict_last are handed back: `applypriority ... L2::evict_normal` (SASS
// CCTL.E.DML2) on every 128-byte line of a row, so that kernels running afterwards find an L2 without 68 MB of lines they cannot
// displace.  `row` .. `row + bytes` is covered from the enclosing 128-byte boundary; one warp per row, lanes stride the lines.
__device__ __forceinline__ void l2_demote_row(const void* row, size_t bytes, int lane)
{
    const uintptr_t first = reinterpret_cast<uintptr_t>(row) & ~(uintptr_t)127, last = reinterpret_cast<uintptr_t>(row) + bytes;
    for (uintptr_t a = first + (uintptr_t)lane * 128; a < last; a += 32 * 128)
        asm volatile("applypriority.global.L2::evict_normal [%0], 128;" ::"l"(a) : "memory");
}

}  // namespace mp
