// mp_signs_many.cu -- the paper's Fig. 1 experiment in the paper's own representation (both items at once):
// P independent problems, each with its OWN Bernoulli dictionary psi_nm = +-1/sqrt(N) (Eq. 13) given as one sign bit per
// entry.  At M = 1000 a packed dictionary is N*M/8 <= 125 KB: it fits in the shared memory of ONE SM, so one CTA owns a problem
// for the whole solve -- no cluster, no grid barrier, no L2 traffic for the dictionary at all; 148 problems run side by side and
// CTAs draw problems from a device counter.
//
// Correlation by table lookup ("four Russians"): once per iteration the CTA builds, for every group of four residual values,
// the 16 signed sums   T[g][nib] = sum_{k<4} (nib_k ? -r_{4g+k} : +r_{4g+k})   (N/4 x 16 floats, 16 KB at N = 1000, fp32 adds in
// ascending k).  Then lane = atom:  c_m = scale * sum_g T[g][nibble_g(bits_m)]  -- one shift, one mask, one shared-memory load and
// one add per FOUR entries instead of a test and a conditional add per entry.  All lanes of a warp read the same 64-byte table row
// (16 distinct banks), so the loads are conflict-free whatever the nibbles are.
//
// Everything else is the contract of mp_recover_signs / mp_recover: fp32 sums of the fp32 rounding of a float64 residual, packed-key
// argmax with the lowest index on ties, float64 residual update (psi_i re-expanded from its bits) with the direct-sum norm, stop
// test on the device, x~ accumulated in float64 (shared memory).
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kSmThreads = 512;
constexpr int kSmWarps = kSmThreads / 32;

struct SignManyParams {
    const uint32_t* bits;       // problem q: bits + q*pstride, [M][ldw] words, bit k of word w = 1 iff Psi[32 w + k][m] < 0
    const float* Y;
    float* X;
    float* R;
    int* n_iter;
    int* idx_trace;
    float* c_trace;
    unsigned int* counter;
    int64_t ldw, pstride, ldy, ldt;
    int N, M, P, Nr, NW, pitch; // NW = ceil(N/32) words per atom, pitch = odd row pitch of the shared-memory copy
    int AG, WP;                 // atom groups of 32, word parts per atom (WP > 1 only when there are fewer groups than warps)
    float scale, eps;
    int max_iter;
};

__global__ void __launch_bounds__(kSmThreads, 1)
mp_many_signs_kernel(const SignManyParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    double* r64 = reinterpret_cast<double*>(smem_raw);                          // Nr doubles (master residual)
    double* xs = r64 + p.Nr;                                                    // M doubles (x~, Eq. 10)
    double* red = xs + ((p.M + 1) & ~1);                                        // per-warp partial sums
    unsigned long long* wkey = reinterpret_cast<unsigned long long*>(red + kSmWarps);
    int* next_p = reinterpret_cast<int*>(wkey + kSmWarps);                      // [4]
    float* r32 = reinterpret_cast<float*>(next_p + 4);                          // Nr floats
    float* lut = r32 + p.Nr;                                                    // [Nr/4][16] signed sums of four residual values
    float* part = lut + 4 * p.Nr;                                               // [M][WP] partial correlations (WP > 1 only)
    uint32_t* sbits = reinterpret_cast<uint32_t*>(part + (p.WP > 1 ? (size_t)p.M * p.WP : 0));   // [M][pitch], stationary

    const int n_items = p.AG * p.WP;
    const double dscale = (double)p.scale;

    for (;;) {
        if (tid == 0) *next_p = (int)atomicAdd(p.counter, 1u);
        __syncthreads();
        const int prob = *next_p;
        if (prob >= p.P) break;
        const uint32_t* bits = p.bits + (int64_t)prob * p.pstride;
        const float* y = p.Y + (int64_t)prob * p.ldy;

        // ---- the problem's dictionary: global -> shared, once ---------------------------------------------------------------
        for (int a = warp; a < p.M; a += kSmWarps)
            for (int w = lane; w < p.NW; w += 32) sbits[(size_t)a * p.pitch + w] = __ldg(bits + (int64_t)a * p.ldw + w);
        // ---- Eq. 8: r <- y, x~ <- 0, ||y||^2 --------------------------------------------------------------------------------------
        double ss = 0.0;
        for (int n = tid; n < p.Nr; n += kSmThreads) {
            const float v = n < p.N ? y[n] : 0.f;
            r64[n] = (double)v;
            r32[n] = v;
            ss += (double)v * (double)v;
        }
        for (int m = tid; m < p.M; m += kSmThreads) xs[m] = 0.0;
        ss = warp_sum(ss);
        if (lane == 0) red[warp] = ss;
        __syncthreads();
        double rr = 0.0;
#pragma unroll
        for (int w = 0; w < kSmWarps; w++) rr += red[w];
        const double thresh2 = ((double)p.eps * (double)p.eps) * rr;
        int t = 0;
        // ---- the loop: while ||r|| > eps ||y|| and t < T ---------------------------------------------------------------
        while ((rr > thresh2) && (t < p.max_iter)) {
            // ---------- table of the 16 signed sums of every four residual values -----------------------------------------------
            for (int e = tid; e < 4 * p.Nr; e += kSmThreads) {
                const int g = e >> 4, nib = e & 15;
                const float4 v = reinterpret_cast<const float4*>(r32)[g];
                float s = (nib & 1) ? -v.x : v.x;
                s += (nib & 2) ? -v.y : v.y;
                s += (nib & 4) ? -v.z : v.z;
                s += (nib & 8) ? -v.w : v.w;
                lut[e] = s;
            }
            __syncthreads();
            // ---------- Eq. 9: lane = atom, one table row per nibble of its bits ---------------------------------------------------
            unsigned long long best = 0ull;
            for (int it = warp; it < n_items; it += kSmWarps) {
                const int g = it / p.WP, q = it - g * p.WP;
                const int a = g * 32 + lane;
                const int w0 = (int)(((int64_t)q * p.NW) / p.WP), w1 = (int)(((int64_t)(q + 1) * p.NW) / p.WP);
                const uint32_t* row = sbits + (size_t)(a < p.M ? a : p.M - 1) * p.pitch;
                float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;
                for (int w = w0; w < w1; w++) {
                    const uint32_t word = row[w];
                    const char* tb = reinterpret_cast<const char*>(lut + 128 * w);     // 8 rows of 16 floats
                    c0 += *reinterpret_cast<const float*>(tb + 0 * 64 + ((word << 2) & 0x3Cu));
                    c1 += *reinterpret_cast<const float*>(tb + 1 * 64 + ((word >> 2) & 0x3Cu));
                    c2 += *reinterpret_cast<const float*>(tb + 2 * 64 + ((word >> 6) & 0x3Cu));
                    c3 += *reinterpret_cast<const float*>(tb + 3 * 64 + ((word >> 10) & 0x3Cu));
                    c0 += *reinterpret_cast<const float*>(tb + 4 * 64 + ((word >> 14) & 0x3Cu));
                    c1 += *reinterpret_cast<const float*>(tb + 5 * 64 + ((word >> 18) & 0x3Cu));
                    c2 += *reinterpret_cast<const float*>(tb + 6 * 64 + ((word >> 22) & 0x3Cu));
                    c3 += *reinterpret_cast<const float*>(tb + 7 * 64 + ((word >> 26) & 0x3Cu));
                }
                const float c = (c0 + c1) + (c2 + c3);
                if (p.WP > 1) {
                    if (a < p.M) part[(size_t)a * p.WP + q] = c;
                } else if (a < p.M) {
                    const unsigned long long k = pack_key(p.scale * c, a);
                    best = k > best ? k : best;
                }
            }
            if (p.WP > 1) {                                                     // few atoms: the word parts are added in ascending order
                __syncthreads();
                for (int a = tid; a < p.M; a += kSmThreads) {
                    float c = part[(size_t)a * p.WP];
                    for (int q = 1; q < p.WP; q++) c += part[(size_t)a * p.WP + q];
                    const unsigned long long k = pack_key(p.scale * c, a);
                    best = k > best ? k : best;
                }
            }
            best = warp_max_redux(best);
            if (lane == 0) wkey[warp] = best;
            __syncthreads();
            const unsigned long long key = warp_max_redux(lane < kSmWarps ? wkey[lane] : 0ull);
            const int i = key_index(key);
            const float c = key_value(key);
            const double cd = (double)c;
            // ---------- Eq. 11 with psi_i[n] = +-scale from the bits of atom i, Eq. 18 direct sum -------------------------------
            {
                const uint32_t* bi = sbits + (size_t)i * p.pitch;
                double s2 = 0.0;
                for (int n = tid; n < p.N; n += kSmThreads) {
                    const uint32_t word = bi[n >> 5];
                    const double psi = ((word >> (n & 31)) & 1u) ? -dscale : dscale;
                    const double v = r64[n] - cd * psi;
                    r64[n] = v;
                    r32[n] = (float)v;
                    s2 += v * v;
                }
                s2 = warp_sum(s2);
                if (lane == 0) red[warp] = s2;
            }
            if (tid == kSmThreads - 32) {
                xs[i] += cd;
                if (p.idx_trace) p.idx_trace[(int64_t)prob * p.ldt + t] = i;
                if (p.c_trace) p.c_trace[(int64_t)prob * p.ldt + t] = c;
            }
            __syncthreads();
            rr = 0.0;
#pragma unroll
            for (int w = 0; w < kSmWarps; w++) rr += red[w];
            t += 1;
        }
        // ---- P:86 return x~, r, t -------------------------------------------------------------------------------------------------
        for (int m = tid; m < p.M; m += kSmThreads) p.X[(int64_t)prob * p.M + m] = (float)xs[m];
        for (int n = tid; n < p.N; n += kSmThreads) p.R[(int64_t)prob * p.N + n] = r32[n];
        if (tid == 0) p.n_iter[prob] = t;
        __syncthreads();                                                        // next_p, xs, sbits are rewritten for the next problem
    }
}

static bool signs_many_plan(int N, int M, const DeviceInfo& di, SignManyParams* p, size_t* smem)
{
    const int NW = (N + 31) / 32;
    const int pitch = NW | 1;
    const int AG = (M + 31) / 32;
    int WP = AG >= kSmWarps ? 1 : kSmWarps / AG;
    if (WP > NW) WP = NW;
    const size_t Nr = (size_t)round_up(N, 128);
    const size_t s = Nr * 8 + 8 * (size_t)round_up(M, 2) + 8 * 2 * kSmWarps + 16 + Nr * 4 + 16 * Nr + (WP > 1 ? 4 * (size_t)M * WP : 0) +
                     4 * (size_t)M * pitch + 64;
    if (s > (size_t)di.smem_optin) return false;
    p->NW = NW; p->pitch = pitch; p->AG = AG; p->WP = WP; p->Nr = (int)Nr;
    *smem = s;
    return true;
}

}  // namespace mp

using namespace mp;

extern "C" {

MP_API size_t mp_workspace_bytes_signs_many(int N, int M, int P)
{
    if (N < 1 || M < 1 || P < 1) return 0;
    return 256;
}

MP_API mp_status mp_recover_signs_many(const uint32_t* bits, int N, int M, int64_t ldw, int64_t problem_stride, float scale,
                                       const float* Y, int64_t ldy, int P, float eps, int max_iter,
                                       float* X, float* R, int* n_iter, int* idx_trace, float* c_trace, int64_t ldt,
                                       void* workspace, size_t workspace_bytes, void* stream)
{
    if (!bits || !Y || !X || !R || !n_iter) return fail(MP_ERR_INVALID_ARG, "bits, Y, X, R and n_iter must be non-null");
    if (N < 1 || M < 1 || P < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1, M >= 1, P >= 1 (got N=%d, M=%d, P=%d)", N, M, P);
    if (ldw < (N + 31) / 32) return fail(MP_ERR_INVALID_ARG, "need ldw >= ceil(N/32) (got %lld)", (long long)ldw);
    if (problem_stride != 0 && problem_stride < (int64_t)M * ldw)
        return fail(MP_ERR_INVALID_ARG, "problem_stride must be 0 (one shared dictionary) or >= M*ldw words");
    if (ldy < N) return fail(MP_ERR_INVALID_ARG, "need ldy >= N");
    if (!(scale > 0.0f)) return fail(MP_ERR_INVALID_ARG, "scale must be > 0");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    if ((idx_trace || c_trace) && ldt < max_iter) return fail(MP_ERR_INVALID_ARG, "need ldt >= max_iter");
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < 256)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= 256 bytes (got %zu)", workspace_bytes);
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    SignManyParams p;
    size_t smem = 0;
    if (!signs_many_plan(N, M, di, &p, &smem))
        return fail(MP_ERR_UNSUPPORTED, "N=%d, M=%d: a packed dictionary (N*M/8 bytes) plus the lookup table does not fit in one SM's shared memory", N, M);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    static thread_local int attr_dev = -1;
    if (attr_dev != di.device) {
        MP_CUDA(cudaFuncSetAttribute(mp_many_signs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        attr_dev = di.device;
    }
    int occ = 0;
    MP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mp_many_signs_kernel, kSmThreads, smem));
    if (occ < 1) return fail(MP_ERR_UNSUPPORTED, "the sign-packed many-problem kernel does not fit on an SM");
    MP_CUDA(cudaMemsetAsync(workspace, 0, 256, s));
    p.bits = bits; p.Y = Y; p.X = X; p.R = R; p.n_iter = n_iter; p.idx_trace = idx_trace; p.c_trace = c_trace;
    p.counter = static_cast<unsigned int*>(workspace);
    p.ldw = ldw; p.pstride = problem_stride; p.ldy = ldy; p.ldt = ldt;
    p.N = N; p.M = M; p.P = P;
    p.scale = scale; p.eps = eps; p.max_iter = max_iter;
    int64_t grid = (int64_t)di.sm_count * occ;
    if (grid > P) grid = P;
    mp_many_signs_kernel<<<(int)grid, kSmThreads, smem, s>>>(p);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

}  // extern "C"
