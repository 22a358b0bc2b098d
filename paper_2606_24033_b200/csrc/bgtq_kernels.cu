// bgtq_kernels.cu -- block-energy reduction (a1), device allocator (a2), quantize-on-append (a4).
// Hand-written CUDA for sm_100a.  Shares nothing with oracle/.
#include <cooperative_groups.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <mutex>
#include <string>

#include "bgtq_internal.h"

namespace bgtq {

#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

// ============================================================================ a1: block energy
// Eq. 4: two plain means of squared block norms, ONE cooperative launch.  Phase 1 streams the activations
// once (HBM-bound, 16-byte loads, fp32 partial sums over <= ~N/512 tokens per column), phase 2 (after a grid-wide barrier)
// reduces the partials in fp64 in a fixed order and applies the score kind.
constexpr int kEnergyMaxChunks = 512;
constexpr int kEnergyThreads = 256;

__device__ __forceinline__ void load8(const float *p, float v[8])
{
    float4 a = __ldg(reinterpret_cast<const float4 *>(p));
    float4 b = __ldg(reinterpret_cast<const float4 *>(p) + 1);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
__device__ __forceinline__ void load8(const __nv_bfloat16 *p, float v[8])
{
    uint4 a = __ldg(reinterpret_cast<const uint4 *>(p));
    uint32_t w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        v[2 * i] = __uint_as_float(w[i] << 16);
        v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
}

// one work item of pass 1: token chunk c of a tensor with rows of row_elems elements, column slab `slab`
template <typename T>
__device__ __forceinline__ void energy_partial_item(const T *__restrict__ x, int64_t n, int row_elems, int n_chunks, int c,
                                                    int slab, float *__restrict__ partial, float *red)
{
    // A row (one token, all heads) is row_elems/8 threads wide; when that is narrower than the CTA the spare
    // threads take other tokens of the chunk (token lanes) and a fixed-order shared-memory reduction joins them.
    const int row_threads = row_elems / 8;
    const int ct = row_threads < kEnergyThreads ? row_threads : kEnergyThreads;   // column threads in this CTA
    const int TS = kEnergyThreads / ct;                                            // token lanes
    const int tsub = threadIdx.x / ct, cidx = threadIdx.x % ct;
    const int col0 = (slab * ct + cidx) * 8;
    const bool active = tsub < TS && col0 < row_elems;
    const int64_t per = (n + n_chunks - 1) / n_chunks;
    const int64_t t_lo = c * per, t_hi = min(n, t_lo + per);
    float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (active) {
        const int64_t step = (int64_t)TS * row_elems;
        const T *p = x + (t_lo + tsub) * row_elems + col0;
        int64_t t = t_lo + tsub;
        for (; t + 3 * TS < t_hi; t += 4 * TS) {      // four independent 16/32-byte loads in flight per thread
            float v[4][8];
#pragma unroll
            for (int u = 0; u < 4; ++u) load8(p + u * step, v[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[e] = fmaf(v[u][e], v[u][e], acc[e]);
            p += 4 * step;
        }
        for (; t < t_hi; t += TS) {
            float v[8];
            load8(p, v);
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[e] = fmaf(v[e], v[e], acc[e]);
            p += step;
        }
    }
    if (TS > 1) {
        __syncthreads();                               // (red may still be read by the previous item)
#pragma unroll
        for (int e = 0; e < 8; ++e) red[threadIdx.x * 8 + e] = acc[e];
        __syncthreads();
        if (tsub == 0 && active) {
            for (int s2 = 1; s2 < TS; ++s2)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[e] += red[(s2 * ct + cidx) * 8 + e];
        }
    }
    if (tsub == 0 && active) {
        float *o = partial + (int64_t)c * row_elems + col0;
        reinterpret_cast<float4 *>(o)[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        reinterpret_cast<float4 *>(o)[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
    }
}

struct EnergyParams {
    const void *q, *k;                 // k: the keys, or the values for the V-side score (v_mode)
    int64_t n_q, n_k;
    int rq, rk, cq, ck, sq, sk;        // row elements, token chunks, column slabs per chunk
    float *pq, *pk;
    int Hq, Hkv, d_h, pairing, kind, v_mode;
    float *scores, *eq_out, *ek_out;
};

// ONE launch (cooperative: all CTAs are resident).  Phase 1: the work items (tensor, token chunk, column slab) of q and k
// are dealt round-robin to the CTAs; grid-wide barrier; phase 2: output (kv head, block) o is reduced by CTA o mod grid
// from the partials in fp64, in a fixed order, and the score kind is applied.
template <typename T>
__global__ void __launch_bounds__(kEnergyThreads)
energy_kernel(const EnergyParams P)
{
    __shared__ float red[kEnergyThreads * 8];
    const int items_q = P.n_q > 0 ? P.cq * P.sq : 0, items_k = P.n_k > 0 ? P.ck * P.sk : 0;
    // the large tensor first: its items are the long ones
    for (int it = blockIdx.x; it < items_q + items_k; it += gridDim.x) {
        if (it < items_k) energy_partial_item<T>((const T *)P.k, P.n_k, P.rk, P.ck, it / P.sk, it % P.sk, P.pk, red);
        else { const int j = it - items_k; energy_partial_item<T>((const T *)P.q, P.n_q, P.rq, P.cq, j / P.sq, j % P.sq, P.pq, red); }
    }
    __threadfence();
    cooperative_groups::this_grid().sync();
    double *s1 = reinterpret_cast<double *>(red), *s2 = s1 + kEnergyThreads;
    const int d_h = P.d_h, L = d_h / 2, G = P.v_mode ? 1 : P.Hq / P.Hkv;
    const int nb = P.v_mode ? d_h / BGTQ_V_BLOCK : L;
    for (int o = blockIdx.x; o < P.Hkv * nb; o += gridDim.x) {
        const int h = o / nb, i = o % nb;
        double sq = 0.0, sk = 0.0;
        if (P.v_mode) {
            for (int c = threadIdx.x; c < P.ck; c += kEnergyThreads) {
                const float *row = P.pk + ((int64_t)c * P.Hkv + h) * d_h + BGTQ_V_BLOCK * i;
#pragma unroll
                for (int u = 0; u < BGTQ_V_BLOCK; ++u) sk += (double)__ldcg(row + u);
            }
        } else {
            const int a = P.pairing == BGTQ_PAIR_HALF ? i : 2 * i;
            const int b = P.pairing == BGTQ_PAIR_HALF ? i + L : 2 * i + 1;
            if (P.n_q > 0)
                for (int c = threadIdx.x; c < P.cq; c += kEnergyThreads)
                    for (int g = h * G; g < h * G + G; ++g) {
                        const float *row = P.pq + ((int64_t)c * P.Hq + g) * d_h;
                        sq += (double)__ldcg(row + a) + (double)__ldcg(row + b);
                    }
            if (P.n_k > 0)
                for (int c = threadIdx.x; c < P.ck; c += kEnergyThreads) {
                    const float *row = P.pk + ((int64_t)c * P.Hkv + h) * d_h;
                    sk += (double)__ldcg(row + a) + (double)__ldcg(row + b);
                }
        }
#pragma unroll
        for (int w = 16; w > 0; w >>= 1) { sq += __shfl_xor_sync(0xffffffffu, sq, w); sk += __shfl_xor_sync(0xffffffffu, sk, w); }
        __syncthreads();
        if ((threadIdx.x & 31) == 0) { s1[threadIdx.x >> 5] = sq; s2[threadIdx.x >> 5] = sk; }
        __syncthreads();
        if (threadIdx.x == 0) {
            sq = 0.0; sk = 0.0;
            for (int w = 0; w < kEnergyThreads / 32; ++w) { sq += s1[w]; sk += s2[w]; }
            s1[0] = sq; s2[0] = sk;
        }
        if (threadIdx.x == 0) {
            if (P.v_mode) { P.scores[o] = (float)(s2[0] / (double)P.n_k); continue; }
            const double eq = P.n_q > 0 ? s1[0] / ((double)P.n_q * (double)G) : 0.0;
            const double ek = P.n_k > 0 ? s2[0] / (double)P.n_k : 0.0;
            double s;
            switch (P.kind) {
            case BGTQ_QK_AVG: s = 0.5 * (eq + ek); break;
            case BGTQ_QK_MAX: s = eq > ek ? eq : ek; break;
            case BGTQ_QK_PRODUCT: s = sqrt(eq * ek); break;
            case BGTQ_K_ONLY: s = ek; break;
            default: s = eq; break;
            }
            P.scores[o] = (float)s;
            if (P.eq_out) P.eq_out[o] = (float)eq;
            if (P.ek_out) P.ek_out[o] = (float)ek;
        }
    }
}

size_t block_energy_ws_bytes(int Hq, int Hkv, int d_h)
{
    return (size_t)kEnergyMaxChunks * (size_t)(Hq + Hkv) * d_h * sizeof(float);
}

static int energy_chunks(int64_t n, int row_elems, int max_chunks = kEnergyMaxChunks)
{
    // a chunk gives each of its threads four tokens (one round of four loads in flight); more tokens per chunk only when
    // the chunk count is capped.  Wide rows (queries: one thread column per 8 elements, no token lanes) get short chunks,
    // so a few hundred calibration tokens still spread over the whole GPU instead of eight CTAs walking 32 rows each.
    const int row_threads = row_elems / 8;
    const int ct = row_threads < kEnergyThreads ? (row_threads > 0 ? row_threads : 1) : kEnergyThreads;
    const int min_per = 4 * (kEnergyThreads / ct);
    int64_t c = (n + min_per - 1) / min_per;
    if (c > max_chunks) c = max_chunks;
    if (c < 1) c = 1;
    // make every chunk non-empty: per = ceil(n/c) tokens, chunks = ceil(n/per)
    if (n > 0) { int64_t per = (n + c - 1) / c; c = (n + per - 1) / per; }
    return (int)c;
}

static int launch_energy(EnergyParams &P, int dt, cudaStream_t st, int max_chunks = kEnergyMaxChunks)
{
    static int blocks_per_sm[64][2] = {};          // occupancy of the two instantiations per device (cooperative grid size)
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int ti = dt == BGTQ_F32 ? 0 : 1;
    if (dev < 64 && blocks_per_sm[dev][ti] == 0) {
        int nb = 0;
        if (ti == 0) CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, energy_kernel<float>, kEnergyThreads, 0));
        else CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, energy_kernel<__nv_bfloat16>, kEnergyThreads, 0));
        blocks_per_sm[dev][ti] = nb < 1 ? 1 : (nb > 4 ? 4 : nb);
    }
    P.cq = energy_chunks(P.n_q, P.rq, max_chunks); P.ck = energy_chunks(P.n_k, P.rk, max_chunks);
    P.sq = (P.rq / 8 + kEnergyThreads - 1) / kEnergyThreads;       // narrow rows: one slab, spare threads take tokens
    P.sk = (P.rk / 8 + kEnergyThreads - 1) / kEnergyThreads;
    if (P.sq < 1) P.sq = 1;
    if (P.sk < 1) P.sk = 1;
    const int items = (P.n_q > 0 ? P.cq * P.sq : 0) + (P.n_k > 0 ? P.ck * P.sk : 0);
    const int outs = P.Hkv * (P.v_mode ? P.d_h / BGTQ_V_BLOCK : P.d_h / 2);
    int grid = sms * (dev < 64 ? blocks_per_sm[dev][ti] : 1);
    const int want = items > outs ? items : outs;
    if (grid > want) grid = want;
    void *args[] = {&P};
    if (dt == BGTQ_F32) CUDA_TRY(cudaLaunchCooperativeKernel((const void *)energy_kernel<float>, dim3(grid), dim3(kEnergyThreads), args, 0, st));
    else CUDA_TRY(cudaLaunchCooperativeKernel((const void *)energy_kernel<__nv_bfloat16>, dim3(grid), dim3(kEnergyThreads), args, 0, st));
    count_launch();
    return BGTQ_OK;
}

int launch_block_energy(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt, int Hq,
                        int Hkv, int d_h, int pairing, int kind, float *scores, float *eq_out,
                        float *ek_out, void *ws, size_t, cudaStream_t st)
{
    EnergyParams P = {};
    P.q = q; P.k = k; P.n_q = n_q; P.n_k = n_k; P.rq = Hq * d_h; P.rk = Hkv * d_h;
    P.pq = (float *)ws; P.pk = P.pq + (size_t)kEnergyMaxChunks * Hq * d_h;
    P.Hq = Hq; P.Hkv = Hkv; P.d_h = d_h; P.pairing = pairing; P.kind = kind; P.v_mode = 0;
    P.scores = scores; P.eq_out = eq_out; P.ek_out = ek_out;
    return launch_energy(P, dt, st);
}

// ---- bgtq_block_energy_static: the same kernel with its partial sums in a file-scope device array instead of a caller
// workspace, for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
// 4 MiB per GPU that loads the library, held until exit.  Every call uses the SAME array: calls that overlap on the GPU
// (different streams, or graphs replayed concurrently) race.  Nothing in it has to start at zero -- phase 2 reads exactly the
// entries phase 1 of the same call has written (every chunk < cq / ck, every column), so stale contents are never read.
constexpr int kStaticEnergyChunks = 128;                                  // token chunks per tensor (the workspace path: 512)
constexpr int kStaticEnergyRowElems = 8192;                               // (n_q_heads + n_kv_heads) * d_h at most
constexpr size_t kStaticEnergyFloats = (size_t)kStaticEnergyChunks * kStaticEnergyRowElems;   // 1,048,576 floats = 4 MiB
static __device__ __align__(256) float g_energy_scratch[kStaticEnergyFloats];

int block_energy_static_max_row_elems() { return kStaticEnergyRowElems; }

int launch_block_energy_static(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt, int Hq, int Hkv, int d_h,
                               int pairing, int kind, float *scores, float *eq_out, float *ek_out, cudaStream_t st)
{
    if ((int64_t)(Hq + Hkv) * d_h > kStaticEnergyRowElems) {
        set_error("bgtq_block_energy_static: (n_q_heads + n_kv_heads) * d_h = " + std::to_string((int64_t)(Hq + Hkv) * d_h) +
                  " exceeds the static scratch limit of " + std::to_string(kStaticEnergyRowElems) + " (4 MiB); use bgtq_block_energy with a workspace");
        return BGTQ_EWORKSPACE;
    }
    // device address of the array: in host code `g_energy_scratch` is only a handle, never a pointer a kernel may use.
    // Looked up once per device, with that device current.
    static float *scratch_of[64] = {};
    static std::mutex mu;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    float *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (dev >= 0 && dev < 64 && scratch_of[dev]) scratch = scratch_of[dev];
        else {
            void *ptr = nullptr;
            CUDA_TRY(cudaGetSymbolAddress(&ptr, g_energy_scratch));
            scratch = static_cast<float *>(ptr);
            if (dev >= 0 && dev < 64) scratch_of[dev] = scratch;
        }
    }
    EnergyParams P = {};
    P.q = q; P.k = k; P.n_q = n_q; P.n_k = n_k; P.rq = Hq * d_h; P.rk = Hkv * d_h;
    P.pq = scratch; P.pk = scratch + (size_t)kStaticEnergyChunks * Hq * d_h;
    P.Hq = Hq; P.Hkv = Hkv; P.d_h = d_h; P.pairing = pairing; P.kind = kind; P.v_mode = 0;
    P.scores = scores; P.eq_out = eq_out; P.ek_out = ek_out;
    return launch_energy(P, dt, st, kStaticEnergyChunks);
}

// V-side score (reading Q19): s^V[h][j] = mean_t ||v_t^(j)||^2 over the 16 coordinates of V block j -- the same kernel,
// phase 2 sums the 16 columns of a block.
int launch_v_block_energy(const void *v, int64_t n, int dt, int Hkv, int d_h, float *scores, void *ws, cudaStream_t st)
{
    EnergyParams P = {};
    P.k = v; P.n_k = n; P.rq = d_h; P.rk = Hkv * d_h; P.pq = (float *)ws; P.pk = (float *)ws;
    P.Hq = Hkv; P.Hkv = Hkv; P.d_h = d_h; P.v_mode = 1; P.scores = scores;
    return launch_energy(P, dt, st);
}

// ============================================================================ a2: Alg. 1 on the device
// One warp per head.  Each lane scans blocks lane, lane+32, ...; the warp arg-max
// takes the largest key, ties to the smallest index (Q4).  key = 3/4 * s * 4^-b, exact in fp64.
__global__ void __launch_bounds__(128)
allocate_kernel(const float *__restrict__ scores, int n_heads, int L, int b_min, int b_max, int B,
                uint8_t *__restrict__ bits)
{
    extern __shared__ unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int head = blockIdx.x * 4 + warp;
    double *s = reinterpret_cast<double *>(smem_raw) + (size_t)warp * L;
    uint8_t *b = smem_raw + 4 * (size_t)L * sizeof(double) + (size_t)warp * L;
    if (head >= n_heads) return;
    for (int i = lane; i < L; i += 32) {
        float v = scores[(size_t)head * L + i];
        s[i] = (v > 0.0f && v < INFINITY) ? (double)v : 0.0;   // negative / NaN -> 0 (bgtq.h)
        b[i] = (uint8_t)b_min;
    }
    __syncwarp();
    for (int extra = B - L * b_min; extra > 0; --extra) {
        double bestkey = -1.0;
        int best = 0x7FFFFFFF;
        for (int i = lane; i < L; i += 32) {
            if (b[i] >= b_max) continue;
            double key = 0.75 * scalbn(s[i], -2 * (int)b[i]);
            if (key > bestkey) { bestkey = key; best = i; }       // ascending i: first max kept
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double ok = __shfl_xor_sync(0xFFFFFFFFu, bestkey, o);
            int oi = __shfl_xor_sync(0xFFFFFFFFu, best, o);
            if (ok > bestkey || (ok == bestkey && oi < best)) { bestkey = ok; best = oi; }
        }
        if (best == 0x7FFFFFFF) break;
        if (lane == 0) b[best] += 1;
        __syncwarp();
    }
    for (int i = lane; i < L; i += 32) bits[(size_t)head * L + i] = b[i];
}

int launch_allocate(const float *scores, int n_heads, int L, int b_min, int b_max, int B,
                    uint8_t *bits, cudaStream_t st)
{
    size_t smem = 4 * (size_t)L * (sizeof(double) + 1);
    allocate_kernel<<<(n_heads + 3) / 4, 128, smem, st>>>(scores, n_heads, L, b_min, b_max, B, bits);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

}  // namespace bgtq
