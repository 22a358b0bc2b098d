// bgtq_kernels.cu -- block-energy reduction (a1), device allocator (a2), quantize-on-append (a4).
// Hand-written CUDA for sm_100a.  Shares nothing with oracle/.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "bgtq_internal.h"

namespace bgtq {

#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

// ============================================================================ a1: block energy
// Eq. 4: two plain means of squared block norms.  Pass 1 streams the activations once
// (HBM-bound, 16-byte loads, fp32 partial sums over <= ~N/512 tokens per column), pass 2 reduces the
// partials in fp64 in a fixed order and applies the score kind.
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

template <typename T>
__global__ void __launch_bounds__(kEnergyThreads)
energy_partial_kernel(const T *__restrict__ x, int64_t n, int row_elems, int n_chunks,
                      float *__restrict__ partial)
{
    // A row (one token, all heads) is row_elems/8 threads wide; when that is narrower than the CTA the spare
    // threads take other tokens of the chunk (token lanes) and a fixed-order shared-memory reduction joins them.
    __shared__ float red[kEnergyThreads * 8];
    const int row_threads = row_elems / 8;
    const int ct = row_threads < kEnergyThreads ? row_threads : kEnergyThreads;   // column threads in this CTA
    const int TS = kEnergyThreads / ct;                                            // token lanes
    const int tsub = threadIdx.x / ct, cidx = threadIdx.x % ct;
    const int col0 = (blockIdx.y * ct + cidx) * 8;
    const bool active = tsub < TS && col0 < row_elems;
    const int c = blockIdx.x;
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

// one CTA of 128 threads per (kv head h, block i): fixed-order fp64 reduction of the partials
__global__ void __launch_bounds__(128)
energy_final_kernel(const float *__restrict__ pq, int cq, int64_t n_q, const float *__restrict__ pk,
                    int ck, int64_t n_k, int Hq, int Hkv, int d_h, int pairing, int kind,
                    float *__restrict__ scores, float *__restrict__ eq_out, float *__restrict__ ek_out)
{
    const int L = d_h / 2, G = Hq / Hkv;
    const int h = blockIdx.x / L, i = blockIdx.x % L;
    const int a = pairing == BGTQ_PAIR_HALF ? i : 2 * i;
    const int b = pairing == BGTQ_PAIR_HALF ? i + L : 2 * i + 1;
    double sq = 0.0, sk = 0.0;
    if (n_q > 0)
        for (int c = threadIdx.x; c < cq; c += 128)
            for (int g = h * G; g < h * G + G; ++g) {
                const float *row = pq + ((int64_t)c * Hq + g) * d_h;
                sq += (double)row[a] + (double)row[b];
            }
    if (n_k > 0)
        for (int c = threadIdx.x; c < ck; c += 128) {
            const float *row = pk + ((int64_t)c * Hkv + h) * d_h;
            sk += (double)row[a] + (double)row[b];
        }
    __shared__ double s1[128], s2[128];
    s1[threadIdx.x] = sq;
    s2[threadIdx.x] = sk;
    __syncthreads();
    for (int w = 64; w > 0; w >>= 1) {
        if (threadIdx.x < w) { s1[threadIdx.x] += s1[threadIdx.x + w]; s2[threadIdx.x] += s2[threadIdx.x + w]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double eq = n_q > 0 ? s1[0] / ((double)n_q * (double)G) : 0.0;
        double ek = n_k > 0 ? s2[0] / (double)n_k : 0.0;
        double s;
        switch (kind) {
        case BGTQ_QK_AVG: s = 0.5 * (eq + ek); break;
        case BGTQ_QK_MAX: s = eq > ek ? eq : ek; break;
        case BGTQ_QK_PRODUCT: s = sqrt(eq * ek); break;
        case BGTQ_K_ONLY: s = ek; break;
        default: s = eq; break;
        }
        scores[h * L + i] = (float)s;
        if (eq_out) eq_out[h * L + i] = (float)eq;
        if (ek_out) ek_out[h * L + i] = (float)ek;
    }
}

size_t block_energy_ws_bytes(int Hq, int Hkv, int d_h)
{
    return (size_t)kEnergyMaxChunks * (size_t)(Hq + Hkv) * d_h * sizeof(float);
}

static int energy_chunks(int64_t n)
{
    int64_t c = (n + 31) / 32;
    if (c > kEnergyMaxChunks) c = kEnergyMaxChunks;
    if (c < 1) c = 1;
    // make every chunk non-empty: per = ceil(n/c) tokens, chunks = ceil(n/per)
    if (n > 0) { int64_t per = (n + c - 1) / c; c = (n + per - 1) / per; }
    return (int)c;
}

int launch_block_energy(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt, int Hq,
                        int Hkv, int d_h, int pairing, int kind, float *scores, float *eq_out,
                        float *ek_out, void *ws, size_t, cudaStream_t st)
{
    float *pq = (float *)ws;
    float *pk = pq + (size_t)kEnergyMaxChunks * Hq * d_h;
    const int cq = energy_chunks(n_q), ck = energy_chunks(n_k);
    const int rq = Hq * d_h, rk = Hkv * d_h;
    if (n_q > 0) {
        dim3 grid(cq, (rq / 8 + kEnergyThreads - 1) / kEnergyThreads);   // narrow rows: one slab, spare threads take tokens
        if (dt == BGTQ_F32) energy_partial_kernel<float><<<grid, kEnergyThreads, 0, st>>>((const float *)q, n_q, rq, cq, pq);
        else energy_partial_kernel<__nv_bfloat16><<<grid, kEnergyThreads, 0, st>>>((const __nv_bfloat16 *)q, n_q, rq, cq, pq);
        count_launch();
    }
    if (n_k > 0) {
        dim3 grid(ck, (rk / 8 + kEnergyThreads - 1) / kEnergyThreads);
        if (dt == BGTQ_F32) energy_partial_kernel<float><<<grid, kEnergyThreads, 0, st>>>((const float *)k, n_k, rk, ck, pk);
        else energy_partial_kernel<__nv_bfloat16><<<grid, kEnergyThreads, 0, st>>>((const __nv_bfloat16 *)k, n_k, rk, ck, pk);
        count_launch();
    }
    energy_final_kernel<<<Hkv * (d_h / 2), 128, 0, st>>>(pq, cq, n_q, pk, ck, n_k, Hq, Hkv, d_h, pairing,
                                                         kind, scores, eq_out, ek_out);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

// V-side score (reading Q19): s^V[h][j] = mean_t ||v_t^(j)||^2 over the 16 coordinates of V block j.  Same two passes:
// the streaming pass above, then one CTA per (kv head, block) reduces its 16 columns' partials in fp64, fixed order.
__global__ void __launch_bounds__(128)
energy_final_v_kernel(const float *__restrict__ pv, int cv, int64_t n, int Hkv, int d_h, float *__restrict__ scores)
{
    const int nb = d_h / BGTQ_V_BLOCK;
    const int h = blockIdx.x / nb, j = blockIdx.x % nb;
    double sv = 0.0;
    for (int c = threadIdx.x; c < cv; c += 128) {
        const float *row = pv + ((int64_t)c * Hkv + h) * d_h + BGTQ_V_BLOCK * j;
#pragma unroll
        for (int u = 0; u < BGTQ_V_BLOCK; ++u) sv += (double)row[u];
    }
    __shared__ double s1[128];
    s1[threadIdx.x] = sv;
    __syncthreads();
    for (int w = 64; w > 0; w >>= 1) {
        if (threadIdx.x < w) s1[threadIdx.x] += s1[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) scores[h * nb + j] = (float)(s1[0] / (double)n);
}

int launch_v_block_energy(const void *v, int64_t n, int dt, int Hkv, int d_h, float *scores, void *ws, cudaStream_t st)
{
    float *pv = (float *)ws;
    const int cv = energy_chunks(n), rv = Hkv * d_h;
    dim3 grid(cv, (rv / 8 + kEnergyThreads - 1) / kEnergyThreads);
    if (dt == BGTQ_F32) energy_partial_kernel<float><<<grid, kEnergyThreads, 0, st>>>((const float *)v, n, rv, cv, pv);
    else energy_partial_kernel<__nv_bfloat16><<<grid, kEnergyThreads, 0, st>>>((const __nv_bfloat16 *)v, n, rv, cv, pv);
    energy_final_v_kernel<<<Hkv * (d_h / BGTQ_V_BLOCK), 128, 0, st>>>(pv, cv, n, Hkv, d_h, scores);
    count_launch(2);
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
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
