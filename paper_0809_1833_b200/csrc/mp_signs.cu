// mp_signs.cu -- MP on a sign-packed Bernoulli dictionary ("1-bit sign-packed Bernoulli dictionary
// (Eq. 13) as a bandwidth-reduced variant").  The paper's experiments all use psi_nm = +-1/sqrt(N) (Eq. 13): one bit
// per entry carries the whole dictionary, 32x fewer bytes than fp32 -- CFG3's 256 MiB become 8 MiB, i.e. 57 KB per SM,
// which is loaded into shared memory ONCE and stays there: the iteration no longer touches HBM or L2 for the dictionary
// and is bound by the ALUs (one conditional add per entry) instead of by bandwidth.
//
//   c_m = scale * sum_n s_mn r_n,  s = +-1 (bit = 1 for a negative entry), evaluated by table lookup: once per iteration every
// CTA builds the 16 signed sums T[g][nib] = sum_{k<4} (nib_k ? -r_{4g+k} : r_{4g+k}) of every four residual values (16 N bytes of
// shared memory) and an atom's correlation is the sum of one table entry per nibble of its bits -- a shift, a mask, a conflict-
// free shared-memory load (all lanes read the same 64-byte row) and an add per FOUR entries (the first version spent a test and a
// conditional add per entry: 9.1 us per iteration at CFG3).  Same loop, boundary and arithmetic contract as the fp32 kernels otherwise (fp32 dots
// of the fp32 rounding of a float64 residual, packed-key argmax with lowest index on ties, one grid barrier per
// iteration, float64 residual update and direct-sum norm, device-side stop test).
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kSgnMaxWarps = 32;

struct SignParams {
    const uint32_t* bits;       // [M][ldw] words, bit k of word w = 1 iff Psi[32 w + k][m] < 0
    const float* y;
    float* x;
    float* r;
    int* n_iter;
    int* idx_trace;
    float* c_trace;
    double* x64;
    unsigned long long* ctrl;   // [0] barrier counter, [1..3] rotating key slots
    int64_t ldw;
    int N, M, Nr, NW, pitch;    // NW = ceil(N/32) words per atom, pitch = odd row pitch of the shared-memory copy
    int AG, WP, atoms_max;      // atom groups of 32, word parts, max atoms per CTA
    float scale;                // |psi_nm|
    float eps;
    int max_iter;
};

// Sign bits of a +-scale dictionary: one warp per atom, ballot per 32 entries.  n_bad counts entries whose magnitude is
// not bit-identical to psi_t[0]'s (the dictionary is then not a Bernoulli one and must not be packed).
__global__ void __launch_bounds__(256)
pack_signs_kernel(const float* __restrict__ psi_t, int N, int M, int64_t ld, uint32_t* __restrict__ bits, int64_t ldw,
                  float* __restrict__ scale_out, int* __restrict__ n_bad)
{
    const int lane = threadIdx.x & 31;
    const int m = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (m >= M) return;
    const uint32_t mag0 = __float_as_uint(psi_t[0]) & 0x7FFFFFFFu;
    const float* row = psi_t + (int64_t)m * ld;
    int bad = 0;
    for (int w = 0; w * 32 < N; w++) {
        const int n = w * 32 + lane;
        const uint32_t u = n < N ? __float_as_uint(row[n]) : mag0;
        bad += (u & 0x7FFFFFFFu) != mag0;
        const uint32_t word = __ballot_sync(0xffffffffu, (u >> 31) != 0u);
        if (lane == 0) bits[(int64_t)m * ldw + w] = word;
    }
    for (int w = (N + 31) / 32 + lane; w < ldw; w += 32) bits[(int64_t)m * ldw + w] = 0u;
    bad = (int)warp_sum((float)bad);
    if (lane == 0 && bad) atomicAdd(n_bad, bad);
    if (m == 0 && lane == 0) *scale_out = __uint_as_float(mag0);
}

__global__ void __launch_bounds__(512, 1)
mp_persistent_signs_kernel(const SignParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int THREADS = blockDim.x, W = THREADS >> 5;
    const int G = gridDim.x;

    double* r64 = reinterpret_cast<double*>(smem_raw);                         // Nr doubles (master residual)
    float* r32 = reinterpret_cast<float*>(r64 + p.Nr);                         // Nr floats (fp32 rounding, feeds the dots)
    unsigned long long* wkey = reinterpret_cast<unsigned long long*>(r32 + p.Nr);
    double* red = reinterpret_cast<double*>(wkey + kSgnMaxWarps);
    unsigned long long* skey = reinterpret_cast<unsigned long long*>(red + kSgnMaxWarps);
    float* lut = reinterpret_cast<float*>(skey + 2);                           // [Nr/4][16] signed sums of four residual values
    float* part = lut + 4 * p.Nr;                                              // [atom of this CTA][word part]
    uint32_t* sbits = reinterpret_cast<uint32_t*>(part + (size_t)p.atoms_max * p.WP);   // [atom][pitch], stationary

    const int a0 = (int)(((int64_t)blockIdx.x * p.M) / G);
    const int a1 = (int)(((int64_t)(blockIdx.x + 1) * p.M) / G);
    const int n_atoms = a1 - a0;

    // ---- the CTA's share of the dictionary: global -> shared, once ------------------------------------------------
    for (int e = tid; e < n_atoms * p.NW; e += THREADS) {
        const int a = e / p.NW, w = e - a * p.NW;
        sbits[(size_t)a * p.pitch + w] = p.bits[(int64_t)(a0 + a) * p.ldw + w];
    }
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

    const int n_items = p.AG * p.WP;
    const double dscale = (double)p.scale;
    int t = 0;
    // ---- the loop: while ||r|| > eps ||y|| and t < T -----------------------------------------------------------
    while ((rr > thresh2) && (t < p.max_iter)) {
        // ---------- table of the 16 signed sums of every four residual values -----------------------------------------------
        for (int e = tid; e < 4 * p.Nr; e += THREADS) {
            const int g = e >> 4, nib = e & 15;
            const float4 v = reinterpret_cast<const float4*>(r32)[g];
            float s = (nib & 1) ? -v.x : v.x;
            s += (nib & 2) ? -v.y : v.y;
            s += (nib & 4) ? -v.z : v.z;
            s += (nib & 8) ? -v.w : v.w;
            lut[e] = s;
        }
        __syncthreads();
        // ---------- Eq. 9: lane = atom, the words of one part, one table row per nibble ----------------------------------------
        for (int it = warp; it < n_items; it += W) {
            const int g = it / p.WP, q = it - g * p.WP;
            const int a = g * 32 + lane;
            const int w0 = (int)(((int64_t)q * p.NW) / p.WP), w1 = (int)(((int64_t)(q + 1) * p.NW) / p.WP);
            const uint32_t* row = sbits + (size_t)(a < n_atoms ? a : (n_atoms > 0 ? n_atoms - 1 : 0)) * p.pitch;
            float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;
            for (int w = w0; w < w1; w++) {
                const uint32_t word = row[w];
                const char* tb = reinterpret_cast<const char*>(lut + 128 * w);          // 8 rows of 16 floats
                c0 += *reinterpret_cast<const float*>(tb + 0 * 64 + ((word << 2) & 0x3Cu));
                c1 += *reinterpret_cast<const float*>(tb + 1 * 64 + ((word >> 2) & 0x3Cu));
                c2 += *reinterpret_cast<const float*>(tb + 2 * 64 + ((word >> 6) & 0x3Cu));
                c3 += *reinterpret_cast<const float*>(tb + 3 * 64 + ((word >> 10) & 0x3Cu));
                c0 += *reinterpret_cast<const float*>(tb + 4 * 64 + ((word >> 14) & 0x3Cu));
                c1 += *reinterpret_cast<const float*>(tb + 5 * 64 + ((word >> 18) & 0x3Cu));
                c2 += *reinterpret_cast<const float*>(tb + 6 * 64 + ((word >> 22) & 0x3Cu));
                c3 += *reinterpret_cast<const float*>(tb + 7 * 64 + ((word >> 26) & 0x3Cu));
            }
            if (a < n_atoms) part[(size_t)a * p.WP + q] = (c0 + c1) + (c2 + c3);
        }
        __syncthreads();
        // ---------- c = scale * sum_q (S_q - 2 neg_q) in ascending q, Eq. 16 packed argmax -----------------------------------
        unsigned long long best = 0ull;
        for (int a = tid; a < n_atoms; a += THREADS) {
            float c = part[(size_t)a * p.WP];
            for (int q = 1; q < p.WP; q++) c += part[(size_t)a * p.WP + q];
            const unsigned long long k = pack_key(p.scale * c, a0 + a);
            best = k > best ? k : best;
        }
        best = warp_max_redux(best);
        const unsigned long long key = grid_argmax(best, wkey, skey, p.ctrl, t);        // block -> grid argmax, one grid barrier (mp_common.cuh)
        const int i = key_index(key);
        const float c = key_value(key);
        const double cd = (double)c;

        // ---------- Eq. 11 with psi_i[n] = +-scale from the bits of atom i, Eq. 18 direct sum ------------------------------
        {
            const uint32_t* bi = p.bits + (int64_t)i * p.ldw;
            double s2 = 0.0;
            for (int n = tid; n < p.N; n += THREADS) {
                const uint32_t word = __ldg(bi + (n >> 5));
                const double psi = ((word >> (n & 31)) & 1u) ? -dscale : dscale;
                const double v = r64[n] - cd * psi;
                r64[n] = v;
                r32[n] = (float)v;
                s2 += v * v;
            }
            s2 = warp_sum(s2);
            if (lane == 0) red[warp] = s2;
        }
        if (blockIdx.x == 0 && tid == THREADS - 32) {                          // not the thread every CTA's barrier waits for
            record_step(p.x64, p.idx_trace, p.c_trace, p.ctrl, t, i, c);
        }
        __syncthreads();
        rr = 0.0;
        for (int w = 0; w < W; w++) rr += red[w];
        t += 1;
    }

    if (blockIdx.x == 0) {
        __threadfence();
        __syncthreads();
        for (int m = tid; m < p.M; m += THREADS) p.x[m] = (float)__ldcg(p.x64 + m);
        for (int n = tid; n < p.N; n += THREADS) p.r[n] = r32[n];
        if (tid == 0) *p.n_iter = t;
    }
}

static bool signs_plan(int N, int M, const DeviceInfo& di, SignParams* p, int* W, size_t* smem)
{
    const int G = di.sm_count > 0 ? di.sm_count : 1;
    const int atoms_max = (M + G - 1) / G;
    const int NW = (N + 31) / 32;
    const int pitch = NW | 1;
    const int AG = (atoms_max + 31) / 32;
    int w = 16;
    int WP = AG >= w ? 1 : w / AG;
    if (WP > NW) WP = NW;
    if (WP > 32) WP = 32;
    const size_t Nr = (size_t)round_up(N, 128);
    const size_t s = Nr * 12 + 8 * (2 * kSgnMaxWarps + 2) + 16 * Nr + 4 * (size_t)atoms_max * WP + 4 * (size_t)atoms_max * pitch + 64;
    if (s > (size_t)di.smem_optin) return false;
    p->NW = NW; p->pitch = pitch; p->AG = AG; p->WP = WP; p->atoms_max = atoms_max;
    *W = w; *smem = s;
    return true;
}

}  // namespace mp

using namespace mp;

extern "C" {

MP_API mp_status mp_pack_signs(const float* psi_t, int N, int M, int64_t ld, uint32_t* bits, int64_t ldw,
                               float* scale_out, int* n_bad, void* stream)
{
    if (!psi_t || !bits || !scale_out || !n_bad) return fail(MP_ERR_INVALID_ARG, "psi_t, bits, scale_out and n_bad must be non-null");
    if (N < 1 || M < 1 || ld < N) return fail(MP_ERR_INVALID_ARG, "need N >= 1, M >= 1, ld >= N");
    if (ldw < (N + 31) / 32) return fail(MP_ERR_INVALID_ARG, "need ldw >= ceil(N/32) (got %lld)", (long long)ldw);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    MP_CUDA(cudaMemsetAsync(n_bad, 0, sizeof(int), s));
    pack_signs_kernel<<<(M + 7) / 8, 256, 0, s>>>(psi_t, N, M, ld, bits, ldw, scale_out, n_bad);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

MP_API mp_status mp_recover_signs(const uint32_t* bits, int N, int M, int64_t ldw, float scale,
                                  const float* y, float eps, int max_iter,
                                  float* x, float* r, int* n_iter, int* idx_trace, float* c_trace,
                                  void* workspace, size_t workspace_bytes, void* stream)
{
    if (!bits || !y || !x || !r || !n_iter) return fail(MP_ERR_INVALID_ARG, "bits, y, x, r and n_iter must be non-null");
    if (N < 1 || M < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1 and M >= 1 (got N=%d, M=%d)", N, M);
    if (ldw < (N + 31) / 32) return fail(MP_ERR_INVALID_ARG, "need ldw >= ceil(N/32) (got %lld)", (long long)ldw);
    if (!(scale > 0.0f)) return fail(MP_ERR_INVALID_ARG, "scale must be > 0");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    const size_t need = mp_workspace_bytes(N, M, 1);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    if (!di.coop) return fail(MP_ERR_UNSUPPORTED, "device does not support cooperative launch");
    SignParams p;
    int W = 16;
    size_t smem = 0;
    if (!signs_plan(N, M, di, &p, &W, &smem))
        return fail(MP_ERR_UNSUPPORTED, "N=%d, M=%d: the packed dictionary share does not fit in shared memory", N, M);
    Workspace ws;
    workspace_layout(N, M, 1, workspace, &ws);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    static thread_local int attr_dev = -1;
    if (attr_dev != di.device) {
        MP_CUDA(cudaFuncSetAttribute(mp_persistent_signs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        attr_dev = di.device;
    }
    int occ = 0;
    MP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mp_persistent_signs_kernel, W * 32, smem));
    if (occ < 1) return fail(MP_ERR_UNSUPPORTED, "sign-packed persistent kernel does not fit one CTA per SM");
    MP_CUDA(cudaMemsetAsync(ws.ctrl, 0, 256 + sizeof(double) * (size_t)M, s));
    p.bits = bits; p.y = y; p.x = x; p.r = r; p.n_iter = n_iter; p.idx_trace = idx_trace; p.c_trace = c_trace;
    p.x64 = ws.x64; p.ctrl = ws.ctrl; p.ldw = ldw;
    p.N = N; p.M = M; p.Nr = round_up(N, 128);
    p.scale = scale; p.eps = eps; p.max_iter = max_iter;
    void* args[] = {(void*)&p};
    MP_CUDA(cudaLaunchCooperativeKernel((const void*)mp_persistent_signs_kernel, dim3(di.sm_count), dim3(W * 32), args, smem, s));
    count_launch();
    return MP_OK;
}

}  // extern "C"
