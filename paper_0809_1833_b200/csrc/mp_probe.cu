// mp_probe.cu -- mp_probe_read: a read-only streaming diagnostic, the ceiling the correlation pass (Eq. 9) is measured against
// ("measure a read-only streaming kernel on the box as the achievable ceiling").
//
// It is the item loop of the register-streaming kernel (mp_persistent_ldg.cu) with everything else taken away: one CTA per SM, each
// owning a contiguous share of the buffer, warps taking 8 KiB items round-robin, 16 independent 128-bit ld.global.cg per lane in
// flight, four FMAs per load against a constant instead of the residual; no shared memory, no barrier, no argmax.  Run over a buffer
// that fits in L2 for many passes it gives the L2 -> SM read rate (the roofline of the cache-resident configurations, CFG2 and
// CFG4 <= 64 MiB); over a buffer much larger than L2 it gives the HBM read rate.  The caller times it (CUDA events on `stream`).
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kProbeThreads = 512;
constexpr int kProbeItem4 = 32 * 16;          // float4 per item: 32 lanes x 16 loads = 8 KiB

__global__ void __launch_bounds__(kProbeThreads, 1)
mp_probe_read_kernel(const float4* __restrict__ buf, unsigned long long items_per_cta, int passes, float* sink)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const float4* base = buf + (size_t)blockIdx.x * items_per_cta * kProbeItem4;
    float acc = 0.f;
    for (int p = 0; p < passes; p++) {
        for (unsigned long long it = warp; it < items_per_cta; it += W) {
            const float4* q = base + it * kProbeItem4 + lane;
            float4 v[16];
#pragma unroll
            for (int u = 0; u < 16; u++)
                asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[u].x), "=f"(v[u].y), "=f"(v[u].z), "=f"(v[u].w) : "l"(q + 32 * u));
#pragma unroll
            for (int u = 0; u < 16; u++) {
                acc = fmaf(v[u].x, 1.0001f, acc); acc = fmaf(v[u].y, 0.9999f, acc);
                acc = fmaf(v[u].z, 1.0002f, acc); acc = fmaf(v[u].w, 0.9998f, acc);
            }
        }
    }
    acc = warp_sum(acc);
    if (lane == 0) atomicAdd(sink, acc);      // one atomic per warp at the very end: keeps the loads alive, costs nothing
}

}  // namespace mp

using namespace mp;

extern "C" mp_status mp_probe_read(const void* buf, size_t bytes, int passes, float* sink, unsigned long long* bytes_read, void* stream)
{
    if (!buf || !sink) return fail(MP_ERR_INVALID_ARG, "buf and sink must be non-null");
    if (reinterpret_cast<uintptr_t>(buf) & 15u) return fail(MP_ERR_INVALID_ARG, "buf must be 16-byte aligned");
    if (passes < 1) return fail(MP_ERR_INVALID_ARG, "need passes >= 1 (got %d)", passes);
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    const int G = di.sm_count > 0 ? di.sm_count : 1;
    const unsigned long long items = bytes / ((size_t)G * kProbeItem4 * sizeof(float4));
    if (items < 1) return fail(MP_ERR_INVALID_ARG, "buffer too small: need at least %zu bytes (8 KiB per SM)", (size_t)G * kProbeItem4 * sizeof(float4));
    if (bytes_read) *bytes_read = items * (unsigned long long)G * kProbeItem4 * sizeof(float4) * (unsigned long long)passes;
    mp_probe_read_kernel<<<G, kProbeThreads, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<const float4*>(buf), items, passes, sink);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}
