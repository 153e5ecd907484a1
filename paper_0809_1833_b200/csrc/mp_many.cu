// mp_many.cu -- P independent MP solves of one shape in ONE launch (the paper's Fig. 1 experiment is
// thousands of small solves, 100 trials per (sigma, rho) cell at M = 1000, each with its own random dictionary).
//
// A problem of that size (4NM <= 4 MB) cannot fill 148 SMs: with the grid-wide kernels of mp_persistent_ldg.cu an iteration
// costs one grid barrier (~3 us) however small the dictionary is.  Here ONE THREAD-BLOCK CLUSTER owns a problem:
//
//   * cluster of C CTAs (1, 2, 4, 8 or 16); CTA q owns atoms [qM/C, (q+1)M/C) of the problem's dictionary.  When the slice
//     fits it is copied into shared memory once and stays there for the whole solve (STAT: an iteration then reads the
//     dictionary at shared-memory speed, no L2 / HBM traffic at all); otherwise the rows are streamed from global memory
//     (L2) with 128-bit ld.global.cg, many in flight per lane.
//   * every lane keeps its part of the fp32 residual in REGISTERS (V float4 per lane, N <= 128 V), so a dictionary byte
//     read from shared memory is used once and nothing else competes for the shared-memory port.  The stationary rows
//     are zero-padded to 128 V floats and to a multiple of A rows, so the A*V 128-bit loads of a step are one base register
//     plus immediates, with no predicates; the products are packed FFMA2 (fma.rn.f32x2: two fp32 FMAs per issue slot --
//     at 128 B/clk of shared memory the loop is bound by instruction issue, not by the FMA units); A ~ 16 / V atoms are
//     reduced together by a transposing butterfly (A - 1 + 5 - log2 A shuffles instead of 5 A).
//   * argmax (Eq. 16) = packed 64-bit keys: warp max (two REDUX) -> every warp sends its key to every CTA of the cluster
//     with st.async (DSMEM store that also counts on the destination's mbarrier: data and signal in one message) -> each CTA
//     waits on its own mbarrier until all W*C keys have landed and every warp takes their max.  No block barrier and no
//     cluster barrier in the exchange (~0.3 us, against ~3 us for a grid barrier through L2).  Slots and barriers alternate
//     by t & 1.
//   * Eq. 11 / Eq. 18 / stop test: as the single-signal kernel -- every CTA reads psi_i (4N bytes from L2; DSMEM would make
//     the owner's shared-memory port the bottleneck of a C-way broadcast) and updates its own float64 copy of r, so all
//     CTAs take the same decision with no second barrier.  Eq. 10 accumulates in float64 in the owner's shared memory.
//   * clusters are persistent: they draw problems from a device counter until none is left.
//
// Arithmetic contract = mp_recover's: fp32 FMA dots of the fp32 rounding of a float64 residual, fixed
// reduction order, float64 residual / norms / coefficients, lowest index on ties.
#include <cooperative_groups.h>

#include "mp_common.cuh"
#include "mp_internal.h"

namespace cg = cooperative_groups;

namespace mp {

constexpr int kManyMaxWarps = 8;
constexpr int kManyMaxCluster = 16;
constexpr int kManySlots = kManyMaxWarps * kManyMaxCluster;   // one key per warp of the cluster
constexpr int kManyMaxN = 2048;

struct ManyParams {
    const float* psi_t;
    const float* Y;
    float* X;
    float* R;
    int* n_iter;
    int* idx_trace;
    float* c_trace;
    unsigned int* counter;       // next problem to hand out
    int64_t ld, pstride, ldy, ldt;
    int N, M, P, Npad, Nr, amax;
    float eps;
    int max_iter;
};

__device__ __forceinline__ float4 many_ldg_cg4(const float4* p)
{
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// shared::cluster address of `saddr` (a shared::cta address) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// (The wait is the plain mbarrier.try_wait of mp_common.cuh: with .acquire.cluster ptxas adds a CCTL.IVALL -- an L1
// invalidate worth ~550 cycles per iteration, 14 % of the kernel in the ncu capture -- which the complete_tx mechanism
// does not need: the bytes are counted on the barrier the reader waits on.)
// 8-byte store into another CTA's shared memory that reports its bytes on that CTA's mbarrier: data and signal in one
// message, no cluster-wide barrier (SASS: ST.ASYNC... / SYNCS)
__device__ __forceinline__ void st_async_u64(uint32_t remote_addr, unsigned long long v, uint32_t remote_bar)
{
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.u64 [%0], %1, [%2];"
                 ::"r"(remote_addr), "l"(v), "r"(remote_bar) : "memory");
}
// packed fp32 FMA (SASS FFMA2): acc.{lo,hi} += a.{lo,hi} * b.{lo,hi}, each lane rounded as fmaf
__device__ __forceinline__ void ffma2(unsigned long long& acc, float ax, float ay, float bx, float by)
{
    unsigned long long a, b;
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(ax), "f"(ay));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(bx), "f"(by));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ float sum2(unsigned long long v)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
    return lo + hi;
}
__host__ __device__ constexpr int many_atoms_per_step(int V) { return V <= 1 ? 16 : V <= 2 ? 8 : V <= 4 ? 4 : V <= 8 ? 2 : 1; }

// Sum of the kManyMaxWarps per-warp partials (absent warps hold 0) as a fixed tree: the same value in every thread and CTA.
__device__ __forceinline__ double sum_partials(const double* red)
{
    const double2 a = reinterpret_cast<const double2*>(red)[0], b = reinterpret_cast<const double2*>(red)[1];
    const double2 c = reinterpret_cast<const double2*>(red)[2], d = reinterpret_cast<const double2*>(red)[3];
    return ((a.x + a.y) + (b.x + b.y)) + ((c.x + c.y) + (d.x + d.y));
}

// Sum acc[a] over the 32 lanes for A atoms at once.  While more than one value is alive, a lane with bit `o` set keeps the
// upper half of the values and hands the lower half to its partner (and vice versa), so the count halves with the offset;
// then a plain xor-butterfly.  Returns the total of atom `which` (a function of the lane alone); fixed order -> deterministic.
template <int A>
__device__ __forceinline__ float reduce_atoms(float (&acc)[A], int lane, int& which)
{
    int cnt = A;
    which = 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        if (cnt > 1) {
            const int half = cnt >> 1;
            const bool hi = (lane & o) != 0;
#pragma unroll
            for (int k = 0; k < A / 2; k++) {
                if (k < half) {
                    const float send = hi ? acc[k] : acc[k + half];
                    const float keep = hi ? acc[k + half] : acc[k];
                    acc[k] = keep + __shfl_xor_sync(0xffffffffu, send, o);
                }
            }
            if (hi) which += half;
            cnt = half;
        } else {
            acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], o);
        }
    }
    return acc[0];
}

// Profiling builds (-DMP_MANY_TIMELINE): thread 0 of CTA 0 of the cluster that solves problem 0 accumulates clock64()
// differences per phase and leaves them in the control block (workspace + 64: 8 x u64) -- see profiles/many_r01.md.
#ifdef MP_MANY_TIMELINE
#define MP_STAMP(k)                                                   \
    do {                                                              \
        if (tl_on) { const long long now = clock64(); tl[k] += now - tl_last; tl_last = now; } \
    } while (0)
#else
#define MP_STAMP(k) do {} while (0)
#endif

template <int V, bool STAT>
__global__ void __launch_bounds__(256, 1)
mp_many_kernel(const ManyParams p)
{
    constexpr int A = many_atoms_per_step(V);                                   // atoms per load step (A*V float4 per lane in flight)
    constexpr int S = A > 8 ? A : 8;                                            // atoms per cross-lane reduction
    constexpr int STEPS = S / A;
    constexpr int RS = 32 * V;                                                  // float4 per stationary row (zero-padded)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cluster = cg::this_cluster();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int THREADS = blockDim.x, W = THREADS >> 5;
    const int C = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();

    double* r64 = reinterpret_cast<double*>(smem_raw);                          // Nr doubles (master residual)
    double* xs = r64 + p.Nr;                                                    // amax doubles: x~ of this CTA's atoms (Eq. 10)
    double* red = xs + ((p.amax + 1) & ~1);                                     // per-warp partial sums
    unsigned long long* slots = reinterpret_cast<unsigned long long*>(red + kManyMaxWarps);   // [2][kManySlots] keys of all warps
    uint64_t* kbar = reinterpret_cast<uint64_t*>(slots + 2 * kManySlots);       // [2] mbarriers: keys of iteration parity 0 / 1
    int* next_p = reinterpret_cast<int*>(kbar + 2);                             // [4]
    float* r32 = reinterpret_cast<float*>(next_p + 4);                          // Nr floats (fp32 rounding, feeds the dots)
    float* dict = r32 + p.Nr;                                                   // STAT: amax x Npad floats, this CTA's atoms

    const int a0 = (int)(((int64_t)rank * p.M) / C);
    const int a1 = (int)(((int64_t)(rank + 1) * p.M) / C);
    const int n_atoms = a1 - a0;
    const int n_groups = (n_atoms + S - 1) / S;
    const int n4 = p.Npad >> 2;
    const bool ragged = p.Npad != p.N;
    const int tail_j = n4 - 1;
    auto mask_tail = [&](float4& q) {                                           // N % 4 != 0: up to 3 caller-owned pad floats per row
        const int n = tail_j << 2;
        if (n + 1 >= p.N) q.y = 0.f;
        if (n + 2 >= p.N) q.z = 0.f;
        q.w = 0.f;
    };

    // key slots of absent ranks and partial sums of absent warps stay 0 so that the reductions below have a fixed length
    for (int k = tid; k < 2 * kManySlots; k += THREADS) slots[k] = 0ull;
    if (tid < kManyMaxWarps) red[tid] = 0.0;
    if (tid == 0) {
        mbar_init(kbar, 1);
        mbar_init(kbar + 1, 1);
        mbar_fence_init();
    }
    uint32_t kphase = 0;                                                        // bit b = parity to wait for on kbar[b]
    __syncthreads();

    for (;;) {
        // ---- next problem for this cluster -------------------------------------------------------------------------------
        if (rank == 0 && tid == 0) {
            const int np = (int)atomicAdd(p.counter, 1u);
            for (int q = 0; q < C; q++) *cluster.map_shared_rank(next_p, q) = np;
        }
        cluster.sync();
        const int prob = *next_p;
        if (prob >= p.P) break;
        const float* psi = p.psi_t + (int64_t)prob * p.pstride;
        const float* y = p.Y + (int64_t)prob * p.ldy;

        // ---- STAT: this CTA's atoms into shared memory, once per problem (pad of a ragged row zeroed) -----------------------
        if (STAT) {
            float4* d4 = reinterpret_cast<float4*>(dict);
            const int rows = n_groups * S;                                      // rows >= n_atoms and columns >= n4 are zero
            const int total = rows * RS;
            for (int base = tid; base < total; base += 8 * THREADS) {          // 8 independent 16-byte loads per thread in flight
                float4 q[8];
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    const int idx = base + k * THREADS;
                    const int a = idx / RS, j = idx - a * RS;
                    q[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (a < n_atoms && j < n4) {
                        q[k] = many_ldg_cg4(reinterpret_cast<const float4*>(psi + (int64_t)(a0 + a) * p.ld) + j);
                        if (ragged && j == tail_j) mask_tail(q[k]);
                    }
                }
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    const int idx = base + k * THREADS;
                    if (idx < total) d4[idx] = q[k];
                }
            }
        }
        // ---- Eq. 8: r <- y (float64 master + fp32 copy), x~ <- 0, ||y||^2 -------------------------------------------------------
        double ss = 0.0;
        for (int n = tid; n < p.Nr; n += THREADS) {
            const float v = n < p.N ? y[n] : 0.f;
            r64[n] = (double)v;
            r32[n] = v;
            ss += (double)v * (double)v;
        }
        for (int a = tid; a < n_atoms; a += THREADS) xs[a] = 0.0;
        ss = warp_sum(ss);
        if (lane == 0) red[warp] = ss;
        __syncthreads();
        double rr = sum_partials(red);
        const double thresh2 = ((double)p.eps * (double)p.eps) * rr;               // ||r|| > eps ||y||  <=>  ||r||^2 > eps^2 ||y||^2
        __syncthreads();

        // groups of A atoms are dealt round-robin to the warps; a lane holds V float4 of each of the A rows
        float4 q[A][V];
        int joff[V];                                                            // streamed rows: a lane's float4 offsets, clamped
#pragma unroll                                                                  // into the row (the residual is 0 beyond N)
        for (int v = 0; v < V; v++) joff[v] = v * 32 + lane < n4 ? v * 32 + lane : n4 - 1;
        auto load_step = [&](int grp, int st) {
            if (STAT) {
                const float4* gb = reinterpret_cast<const float4*>(dict) + (grp * S + st * A) * RS + lane;
#pragma unroll
                for (int a = 0; a < A; a++)
#pragma unroll
                    for (int v = 0; v < V; v++) q[a][v] = gb[a * RS + v * 32];
            } else {
#pragma unroll
                for (int a = 0; a < A; a++) {
                    const int at = grp * S + st * A + a;
                    const int rel = at < n_atoms ? at : n_atoms - 1;            // a short last group re-reads its last atom
                    const float4* row = reinterpret_cast<const float4*>(psi + (int64_t)(a0 + rel) * p.ld);
#pragma unroll
                    for (int v = 0; v < V; v++) q[a][v] = many_ldg_cg4(row + joff[v]);
                }
                if (ragged) {
#pragma unroll
                    for (int a = 0; a < A; a++)
#pragma unroll
                        for (int v = 0; v < V; v++)
                            if (joff[v] == tail_j) mask_tail(q[a][v]);
                }
            }
        };
        int g = warp;
        bool have = g < n_groups;
        if (have) load_step(g, 0);
        int t = 0;
#ifdef MP_MANY_TIMELINE
        const bool tl_on = prob == 0 && rank == 0 && tid == 0;
        long long tl[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        long long tl_last = clock64();
#endif
        // ---- the loop: while ||r|| > eps ||y|| and t < T ---------------------------------------------------------------
        while ((rr > thresh2) && (t < p.max_iter)) {
            // ---------- Eq. 9 + Eq. 16 over this CTA's atoms: residual in registers, A atoms per warp step -----------------
            MP_STAMP(7);
            float4 rv[V];
#pragma unroll
            for (int v = 0; v < V; v++) rv[v] = reinterpret_cast<const float4*>(r32)[v * 32 + lane];
            unsigned long long best = 0ull;
            while (have) {                                                      // q holds step 0 of group g
                float acc[S];
                int gc = g;
#pragma unroll
                for (int st = 0; st < STEPS; st++) {
#pragma unroll
                    for (int a = 0; a < A; a++) {                               // four packed chains per atom, added as a tree
                        unsigned long long s0 = 0ull, s1 = 0ull, s2 = 0ull, s3 = 0ull;
#pragma unroll
                        for (int v = 0; v < V; v++) {
                            if (v & 1) {
                                ffma2(s2, q[a][v].x, q[a][v].y, rv[v].x, rv[v].y);
                                ffma2(s3, q[a][v].z, q[a][v].w, rv[v].z, rv[v].w);
                            } else {
                                ffma2(s0, q[a][v].x, q[a][v].y, rv[v].x, rv[v].y);
                                ffma2(s1, q[a][v].z, q[a][v].w, rv[v].z, rv[v].w);
                            }
                        }
                        acc[st * A + a] = V > 1 ? (sum2(s0) + sum2(s1)) + (sum2(s2) + sum2(s3)) : sum2(s0) + sum2(s1);
                    }
                    // the next rows are requested before the shuffles below: the stream never drains
                    if (st + 1 < STEPS) load_step(g, st + 1);
                    else {
                        g += W;
                        have = g < n_groups;
                        if (have) load_step(g, 0);
                    }
                }
                int which;                                                      // ONE 5-stage butterfly per S atoms: the shuffles
                const float c = reduce_atoms<S>(acc, lane, which);              // queue behind the 128-bit loads in the MIO pipe
                if (gc * S + which < n_atoms) {
                    const unsigned long long k = pack_key(c, a0 + gc * S + which);
                    best = k > best ? k : best;
                }
            }
            best = warp_max_redux(best);
            MP_STAMP(0);
            // ---------- every warp sends its key to every CTA of the cluster: one st.async per destination carries the key AND
            // counts on the destination's mbarrier -- no block barrier, no cluster-wide barrier.  The barrier completes when all
            // W*C keys have landed, i.e. when every warp of the cluster has finished reading r; barriers and slots alternate
            // with the parity of t ----------------------------------------------------------------------------------------------
            const int par = t & 1;
            if (lane < C)
                st_async_u64(mapa_u32(smem_u32(slots + par * kManySlots + rank * kManyMaxWarps + warp), lane), best,
                             mapa_u32(smem_u32(kbar + par), lane));
            if (tid == 0) mbar_arrive_expect_tx(kbar + par, 8u * C * W);
            MP_STAMP(2);
            mbar_wait(kbar + par, (kphase >> par) & 1u);                       // completion makes the st.async data visible
            kphase ^= 1u << par;
            MP_STAMP(3);
            unsigned long long key;
            {                                                                   // 128 slots (absent ones hold 0): 4 per lane
                const ulonglong2 u = reinterpret_cast<const ulonglong2*>(slots + par * kManySlots)[lane * 2];
                const ulonglong2 w = reinterpret_cast<const ulonglong2*>(slots + par * kManySlots)[lane * 2 + 1];
                const unsigned long long m0 = u.x > u.y ? u.x : u.y, m1 = w.x > w.y ? w.x : w.y;
                key = warp_max_redux(m0 > m1 ? m0 : m1);
            }
            const int i = key_index(key);
            const float c = key_value(key);
            const double cd = (double)c;

            // ---------- Eq. 11 on this CTA's float64 r, Eq. 18 direct sum ---------------------------------------------------
            {
                const float4* psi4 = reinterpret_cast<const float4*>(psi + (int64_t)i * p.ld);
                float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f);
                if (tid < n4) q0 = __ldg(psi4 + tid);                           // psi_i: 4N bytes from L2, ~0.4 us away
                // The dictionary never changes: the first group of the NEXT iteration is requested now, while psi_i is on its
                // way and the shared-memory port is idle (requested before the exchange it would delay the keys behind it).
                g = warp;
                have = g < n_groups;
                if (have) load_step(g, 0);
                double s2 = 0.0;
                for (int j = tid; j < n4; j += THREADS) {
                    const float4 q = j == tid ? q0 : __ldg(psi4 + j);
                    const int n = j << 2;
                    double v0 = r64[n] - cd * (double)q.x;
                    double v1 = r64[n + 1] - cd * (double)q.y;
                    double v2 = r64[n + 2] - cd * (double)q.z;
                    double v3 = r64[n + 3] - cd * (double)q.w;
                    if (n + 3 >= p.N) {                                         // keep the pad of r at zero
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
            MP_STAMP(4);
            // ---------- Eq. 10 (owner of atom i), Eq. 12, traces (CTA 0) -----------------------------------------------------
            if (tid == THREADS - 32) {                                          // a warp with the least update work
                if (i >= a0 && i < a1) xs[i - a0] += cd;
                if (rank == 0) {
                    if (p.idx_trace) p.idx_trace[(int64_t)prob * p.ldt + t] = i;
                    if (p.c_trace) p.c_trace[(int64_t)prob * p.ldt + t] = c;
                }
            }
            MP_STAMP(5);
            __syncthreads();
            rr = sum_partials(red);
            t += 1;
            MP_STAMP(6);
        }
#ifdef MP_MANY_TIMELINE
        if (tl_on) for (int k = 0; k < 8; k++) reinterpret_cast<long long*>(p.counter)[8 + k] = tl[k];
#endif

        // ---- P:86 return x~ (every CTA its atoms), r and t (CTA 0) ------------------------------------------------------------
        for (int a = tid; a < n_atoms; a += THREADS) p.X[(int64_t)prob * p.M + a0 + a] = (float)xs[a];
        if (rank == 0) {
            for (int n = tid; n < p.N; n += THREADS) p.R[(int64_t)prob * p.N + n] = r32[n];
            if (tid == 0) p.n_iter[prob] = t;
        }
        cluster.sync();                                                         // nobody writes my slots / next_p any more
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Plan.  Measured on B200 (profiles/many_r01.md): with many problems the rate is set by how many dictionaries are in flight --
// as many clusters as possible while their dictionaries together stay L2-resident (~64 MB) stream at 11-13 TB/s; more
// clusters than that fall to the HBM rate (~6.9 TB/s), fewer leave SMs idle.  With few problems the shared-memory-
// stationary variant with the largest cluster wins (2.1 us per iteration at 1 MiB against 3.6 us for the grid-wide kernel).
// So: Qt = min(P, 64 MB / 4NM) problems should be in flight; among (threads, C) whose co-resident cluster count reaches
// ~0.85 Qt take the one that gives a problem the most threads (C * threads), stationary if the slices fit; launch <= Qt
// (+10 %) clusters.
static const int kManyV[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 14, 16};      // float4 per lane; rows are padded to 128 V floats

static size_t many_smem(int Nr, int amax, int V, bool stat)
{
    return (size_t)Nr * 12 + 8 * (size_t)round_up(amax, 2) + 8 * (size_t)(kManyMaxWarps + 2 * kManySlots + 2) + 16 +
           (stat ? (size_t)round_up(amax, many_atoms_per_step(V) > 8 ? many_atoms_per_step(V) : 8) * Nr * 4 : 0) + 16;
}

bool many_supported(int N, int M) { return N <= kManyMaxN && M >= 1; }

// one problem whose dictionary a single cluster can hold in shared memory: the cluster kernel beats the grid-wide ones
bool many_single_stationary(int N, int M)
{
    DeviceInfo di;
    if (!many_supported(N, M) || device_info(&di) != MP_OK) return false;
    const int n4 = round_up(N, 4) / 4;
    int V = 16;
    for (int k = 0; k < (int)(sizeof(kManyV) / sizeof(int)); k++)
        if (32 * kManyV[k] >= n4) { V = kManyV[k]; break; }
    int C = 1;
    while (C < kManyMaxCluster && M / (C * 2) >= 16) C *= 2;
    return many_smem(128 * V, (M + C - 1) / C, V, true) <= (size_t)di.smem_optin;
}

template <int V, bool STAT>
static int many_clusters(int C, int threads, size_t smem)
{
    // co-resident clusters of this configuration (0 = cannot be placed); cached per process and device
    struct Entry { int dev, C, threads; size_t smem; int clusters; };
    static thread_local Entry cache[32];
    static thread_local int n_cache = 0;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    for (int k = 0; k < n_cache; k++)
        if (cache[k].dev == dev && cache[k].C == C && cache[k].threads == threads && cache[k].smem == smem) return cache[k].clusters;
    auto kern = mp_many_kernel<V, STAT>;
    static thread_local int attr_dev = -1;
    if (attr_dev != dev) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)) != cudaSuccess ||
            cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
            (void)cudaGetLastError();
            return 0;
        }
        attr_dev = dev;
    }
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cfg.blockDim = dim3(threads); cfg.gridDim = dim3(C); cfg.dynamicSmemBytes = smem;
    int clusters = 0;
    if (cudaOccupancyMaxActiveClusters(&clusters, kern, &cfg) != cudaSuccess) { (void)cudaGetLastError(); clusters = 0; }
    if (n_cache < 32) cache[n_cache++] = Entry{dev, C, threads, smem, clusters};
    return clusters;
}

template <int V, bool STAT>
static mp_status many_launch(const ManyParams& p, int C, int threads, size_t smem, int n_clusters, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cfg.blockDim = dim3(threads); cfg.gridDim = dim3(n_clusters * C); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    MP_CUDA(cudaLaunchKernelEx(&cfg, mp_many_kernel<V, STAT>, p));
    count_launch();
    options().info_many_cluster = C;
    options().info_many_stat = STAT ? 1 : 0;
    options().info_many_clusters = n_clusters;
    options().info_many_threads = threads;
    return MP_OK;
}

template <int V>
static mp_status many_plan_and_launch(ManyParams p, const DeviceInfo& di, cudaStream_t stream)
{
    const Options& o = options();
    const double bytes = 4.0 * p.N * p.M;
    const double l2_budget = o.many_l2_mb > 0 ? 1e6 * (double)o.many_l2_mb : 64e6;   // dictionaries in flight stay L2-resident
    int64_t qt = p.pstride == 0 ? p.P : (int64_t)(l2_budget / bytes);               // one shared dictionary: its footprint does not grow
    if (qt < 1) qt = 1;
    if (qt > p.P) qt = p.P;
    int c_cap = 1;
    while (c_cap < kManyMaxCluster && p.M / (c_cap * 2) >= 16) c_cap *= 2;      // at least 16 atoms per CTA
    const bool force_c = o.many_cluster == 1 || o.many_cluster == 2 || o.many_cluster == 4 || o.many_cluster == 8 || o.many_cluster == 16;
    const int force_th = o.many_threads >= 32 && o.many_threads <= 256 ? (int)o.many_threads / 32 * 32 : 0;
    int bC = 0, bT = 0, bCl = 0; bool bS = false; size_t bSm = 0; int64_t bScore = -1;
    int fC = 0, fT = 0, fCl = 0; bool fS = false; size_t fSm = 0;             // fallback: most clusters
    const int ths[2] = {256, 128};                                              // ties go to 128 threads (two CTAs per SM) ...
    for (int ti = 0; ti < 2; ti++) {
        const int th = force_th ? force_th : ths[ti];
        if (force_th && ti) break;
        for (int C = kManyMaxCluster; C >= 1; C /= 2) {
            if (force_c ? C != (o.many_cluster <= p.M ? (int)o.many_cluster : 1) : C > c_cap) continue;
            const int amax = (p.M + C - 1) / C;
            for (int st = 1; st >= 0; st--) {
                if (st && (o.many_stat == 2 || (th != 256 && !force_th))) continue;   // stationary: one CTA per SM, all 8 warps
                const size_t sm = many_smem(p.Nr, amax, V, st != 0);
                if (sm > (size_t)di.smem_optin) continue;
                const int cl = st ? many_clusters<V, true>(C, th, sm) : many_clusters<V, false>(C, th, sm);
                if (cl < 1) continue;
                if (cl > fCl) { fC = C; fT = th; fCl = cl; fS = st != 0; fSm = sm; }
                if ((double)cl < 0.85 * (double)qt) continue;
                const int64_t score = (int64_t)C * th * 2 + st;
                if (score > bScore || (score == bScore && C < kManyMaxCluster)) {   // ... except for 16-CTA clusters, which place badly
                    bScore = score; bC = C; bT = th; bCl = cl; bS = st != 0; bSm = sm;
                }
            }
        }
    }
    if (bScore < 0) { bC = fC; bT = fT; bCl = fCl; bS = fS; bSm = fSm; }
    if (bC == 0) return fail(MP_ERR_UNSUPPORTED, "no cluster configuration of the many-problem kernel can be placed (N=%d, M=%d)", p.N, p.M);
    int64_t want = qt + (qt + 9) / 10;                                          // in flight: <= Qt (+10 %)
    if (want > p.P) want = p.P;
    const int n_clusters = (int)(bCl < want ? bCl : want);
    p.amax = (p.M + bC - 1) / bC;
    return bS ? many_launch<V, true>(p, bC, bT, bSm, n_clusters, stream) : many_launch<V, false>(p, bC, bT, bSm, n_clusters, stream);
}

mp_status launch_recover_many(const ManyArgs& a, unsigned int* counter, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    if (!many_supported(a.N, a.M)) return fail(MP_ERR_UNSUPPORTED, "the cluster-per-problem kernel needs N <= %d (got %d)", kManyMaxN, a.N);
    const int n4 = round_up(a.N, 4) / 4;
    int V = 16;
    for (int k = 0; k < (int)(sizeof(kManyV) / sizeof(int)); k++)
        if (32 * kManyV[k] >= n4) { V = kManyV[k]; break; }
    MP_CUDA(cudaMemsetAsync(counter, 0, 256, stream));
    ManyParams p;
    p.psi_t = a.psi_t; p.Y = a.Y; p.X = a.X; p.R = a.R; p.n_iter = a.n_iter; p.idx_trace = a.idx_trace; p.c_trace = a.c_trace;
    p.counter = counter;
    p.ld = a.ld; p.pstride = a.pstride; p.ldy = a.ldy; p.ldt = a.ldt;
    p.N = a.N; p.M = a.M; p.P = a.P; p.Npad = round_up(a.N, 4); p.Nr = 128 * V; p.amax = 0;
    p.eps = a.eps; p.max_iter = a.max_iter;
#define MP_MANY_CASE(v) if (V == v) return many_plan_and_launch<v>(p, di, stream);
    MP_MANY_CASE(1) MP_MANY_CASE(2) MP_MANY_CASE(3) MP_MANY_CASE(4) MP_MANY_CASE(5) MP_MANY_CASE(6) MP_MANY_CASE(7) MP_MANY_CASE(8)
    MP_MANY_CASE(10) MP_MANY_CASE(12) MP_MANY_CASE(14) MP_MANY_CASE(16)
#undef MP_MANY_CASE
    return fail(MP_ERR_UNSUPPORTED, "N=%d does not fit the cluster-per-problem kernel", a.N);
}

}  // namespace mp
