// bgtq_decode2.cu -- split-KV decode attention over a BGTQ-v2 ("row order") packed cache on the 5th-generation tensor
// cores.  Hand-written for sm_100a: tcgen05.mma with the A operand in tensor memory.
//
// Why a second kernel.  The round-1 kernel (bgtq_decode.cu) unpacks codes to fp16 mma.sync fragments: ~46 ALU-pipe
// instructions per 1024 codes, and the ALU pipe (PRMT / LOP3 / SHF, one warp instruction per two clocks per scheduler)
// is what binds it at 37 % of the HBM roofline.  An 8-bit operand needs ONE byte lookup (PRMT) per four codes and plane;
// sm_100a has no fp8 mma.sync (it is emulated through fp16), but tcgen05.mma kind::f8f6f4 takes e4m3 operands natively
// and reads A from tensor memory, where a thread can write the bytes it has just looked up (tcgen05.st) -- no shared
// memory round trip.  Codebook level v of width b is hi[v] + lo[v] in e4m3 (exact for b = 1, 3; see codebook_planes),
// q' and the softmax weights are split into three e4m3 planes, all products accumulate in fp32 in tensor memory.
//
// Algebra: with q'_g = Pi^(m_g) q_g * (scale*log2e / (sqrt(m_g) kappa_g sigma_n)) split as
// q1 + q2 + q3 (e4m3 each), and kappa_g C_g[idx] = hi + lo:
//     log2e*logit_t = sigma_n * sum_g n_{t,g} * S_g[t],   S_g = (hi + lo)(q1 + q2 + q3)  (lo*q3 dropped: 2^-14 relative)
//     P'_t = 2^(logit2_t + log2 h^V_t - R_n) = P1 + 2^-4 P2 + 2^-8 P3   (three e4m3 planes, three accumulators)
//     acc  = sum_t P'_t * (hi^V + lo^V)[idx^V_t] / kappa_V,  l = sum_t P'_t / h^V_t
// R_n is a running reference (not the running maximum): it moves only when a logit would leave the e4m3 range, and then
// the accumulators in tensor memory are rescaled.  The partial record (R_n, l, acc) has the format of the round-1 kernel,
// so the exact log-sum-exp merge and the V de-rotation stay in combine_kernel (a6).
//
// Mapping: one CTA per SM, 14 warps.  Tile = 128 tokens; row r of an operand is TMEM lane r.
//   warps 0-3   K unpack: thread = token row, chunk = 32 coordinates -> 8 columns per plane of A_K (tcgen05.st)
//   warps 4-7   softmax:  thread = token row, S_g read with tcgen05.ld, group norms, planes of P' -> shared memory (B of PV)
//   warps 8-11  V unpack: thread = dimension row, chunk = 32 tokens -> A_V
//   warp 12     one thread issues every tcgen05.mma (QK^T: M=128 tokens, N=8 heads, K=32 per chunk; PV: M=128 dims, N=8, K=32 tokens)
//   warp 13     one thread streams whole tiles into a shared-memory ring with TMA bulk copies (cp.async.bulk + mbarrier)
// Work split: the global tile list [layer][sequence][kv head][tile] is cut into one contiguous range per CTA
// (flash-decoding along the key axis); a CTA writes one partial record per (layer, sequence, head) it touches.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <string>

#include "bgtq_internal.h"
#include "bgtq_device.cuh"

namespace bgtq {

#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

constexpr int kQkIssuers = 4, kPvIssuers = 2;                 // a thread issues one tcgen05.mma per ~60 clocks: several issuers in parallel
constexpr int kD2Warps = 13 + kQkIssuers + kPvIssuers;
constexpr int kD2Threads = kD2Warps * 32;
constexpr int kD2Consumers = (kD2Warps - 1) * 32;             // every warp but the TMA producer (named barrier 1)
constexpr int kQ2Planes = 3;
constexpr int kQ2Atoms = (kQ2Planes * kMaxChunks + 3) / 4;    // (chunk, plane) slices of [8 heads x 32 bytes], four per 1 KB atom
constexpr int kQ2ImageBytes = kQ2Atoms * 1024;
constexpr int kQ2Stride = kQ2ImageBytes + 128;                // + sigma_n (8 floats)
constexpr int kP2Bytes = 3 * 1024;                            // P' planes: 12 slices (4 token quarters x 3 planes) = 3 atoms
constexpr int kMaxStages = 10;
// tensor memory columns (512 allocated).  A_K: 192 columns = one buffer of 12 chunks x (hi, lo) or, when no head has more
// than 6 chunks, two buffers of 6 chunks; A_V, S, P' double-buffered; O: three planes of 8 heads.
constexpr int kColAK = 0, kColAV = 192, kColS = 320, kColO = 448;
constexpr float kRefHeadroom = 5.0f;      // a new reference puts the largest weight at 2^5
constexpr float kRefLimit = 8.5f;         // weights above 2^8.5 (e4m3 max 448) force a new reference

struct Decode2Params {
    const HeadMeta *metas;
    const uint8_t *cache;
    const uint8_t *qimg;        // [pair][kQ2Stride]
    const int32_t *seq_len;
    const uint8_t *planes;      // [2][512] e4m3 planes of the codebooks
    float *partials;            // [n_ctas + 2 * n_pairs][8][130]
    int64_t n_cap;
    int n_layers, batch, Hkv, G;
    int stage_bytes, n_stages;
    int ak_bufs;                // 2 when every head has <= 6 K chunks, else 1
    float inv_kappa_v;
    const int32_t *pages;
    int pstride;
    int64_t n_pages;
    int n_sink, n_recent;
};

// ---------------------------------------------------------------- prologue: q' -> three e4m3 planes in UMMA B-operand order
__device__ __forceinline__ uint32_t cvt_e4m3x2(float lo, float hi)            // bytes: [e4m3(lo), e4m3(hi)]
{
    uint16_t r;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ float2 e4m3x2_to_f32(uint32_t v)
{
    uint32_t h2;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)v));
    return __half22float2(*reinterpret_cast<const __half2 *>(&h2));
}
// byte offset of element (row n, k) of slice sl in a K-major SWIZZLE_128B image of [8 rows x 128 bytes] atoms
__device__ __forceinline__ int sw128_off(int sl, int n, int k)
{
    return (sl >> 2) * 1024 + n * 128 + (((((sl & 3) << 1) | (k >> 4)) ^ n) << 4) + (k & 15);
}

__global__ void __launch_bounds__(128)
qfold2_kernel(const HeadMeta *__restrict__ metas, const float *__restrict__ rot_t, const __nv_bfloat16 *__restrict__ q,
              int batch, int Hkv, int Hq, float scale_log2e, const float *__restrict__ kappa, uint8_t *__restrict__ qimg)
{
    pdl_trigger();
    const int G = Hq / Hkv;
    const int pair = blockIdx.x / G, n = blockIdx.x % G;
    const int h = pair % Hkv, lb = pair / Hkv, l = lb / batch;
    __shared__ __align__(8) HeadMeta Ms;
    __shared__ float qs[kDh];
    __shared__ float wmax[4];
    const int tid = threadIdx.x;
    {
        const uint32_t *msrc = reinterpret_cast<const uint32_t *>(metas + l * Hkv + h);
        if (tid < (int)(sizeof(HeadMeta) / 4)) reinterpret_cast<uint32_t *>(&Ms)[tid] = __ldg(msrc + tid);
    }
    qs[tid] = __bfloat162float(q[((size_t)lb * Hq + h * G + n) * kDh + tid]);
    __syncthreads();
    const HeadMeta &M = Ms;
    uint8_t *img = qimg + (size_t)pair * kQ2Stride;
    // zero this head's row of every atom (and, from block n = 0, the unused head rows n >= G)
    for (int e = tid; e < kQ2Atoms * 8 * 8; e += 128) {               // 16-byte pieces: [atom][row][8]
        const int row = (e >> 3) & 7;
        if (row == n || (n == 0 && row >= G)) reinterpret_cast<uint4 *>(img)[e] = make_uint4(0u, 0u, 0u, 0u);
    }
    float acc = 0.f;
    int ch = 0, kk = 0;
    if (tid < M.kdim) {
        int g = 0;
        while (g + 1 < M.n_groups && tid >= M.gstart[g + 1]) ++g;
        const int m = M.gm[g], x0 = M.gstart[g], r = tid - x0;
        const float *T = rot_t + rot_offset(m) + r;
        const uint8_t *co = M.coords + x0;
        int k = 0;
        for (; k + 16 <= m; k += 16) {
            float tv[16];
#pragma unroll
            for (int u = 0; u < 16; ++u) tv[u] = __ldg(T + (size_t)(k + u) * m);
#pragma unroll
            for (int u = 0; u < 16; ++u) acc = fmaf(tv[u], qs[co[k + u]], acc);
        }
        for (; k < m; ++k) acc = fmaf(__ldg(T + (size_t)k * m), qs[co[k]], acc);
        acc *= scale_log2e / (sqrtf((float)m) * __ldg(kappa + M.gb[g]));
        while (ch + 1 < M.n_ksteps && tid >= M.chunks[ch + 1].ustart) ++ch;
        kk = tid - M.chunks[ch].ustart;
    }
    // sigma_n: a power of two that puts the largest |q'| of this head into [112, 224] (e4m3: finite up to 448)
    float mx = fabsf(acc);
#pragma unroll
    for (int s = 16; s; s >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    if ((tid & 31) == 0) wmax[tid >> 5] = mx;
    __syncthreads();
    mx = fmaxf(fmaxf(wmax[0], wmax[1]), fmaxf(wmax[2], wmax[3]));
    int e2 = 0;
    if (mx > 0.f) { (void)frexpf(mx, &e2); e2 -= 8; }                   // mx = f * 2^e, f in [0.5, 1): mx / 2^(e-8) in [128, 256)
    const float sigma = ldexpf(1.f, e2);
    if (tid == 0) reinterpret_cast<float *>(img + kQ2ImageBytes)[n] = sigma;
    if (n == 0 && tid >= G && tid < 8) reinterpret_cast<float *>(img + kQ2ImageBytes)[tid] = 0.f;
    if (tid < M.kdim) {
        const float y = acc * ldexpf(1.f, -e2);
        const uint32_t b1 = cvt_e4m3x2(y, 0.f) & 0xFF;
        const float r1 = y - e4m3x2_to_f32(b1).x;
        const uint32_t b2 = cvt_e4m3x2(r1, 0.f) & 0xFF;
        const float r2 = r1 - e4m3x2_to_f32(b2).x;
        const uint32_t b3 = cvt_e4m3x2(r2, 0.f) & 0xFF;
        img[sw128_off(3 * ch + 0, n, kk)] = (uint8_t)b1;
        img[sw128_off(3 * ch + 1, n, kk)] = (uint8_t)b2;
        img[sw128_off(3 * ch + 2, n, kk)] = (uint8_t)b3;
    }
    pdl_wait();
}

// ---------------------------------------------------------------- chunk decoders: 32 slots of one row -> 8 + 8 registers of e4m3 bytes
// pools (registers, from shared memory): byte planes hi / lo of the width's levels (codebook_planes).
struct Pools2 {
    uint32_t hi2, lo2;                  // b = 2: levels 0..3
    uint32_t hi3a, hi3b, lo3a, lo3b;    // b = 3: levels 0..3, 4..7
    uint32_t hi4a, hi4b, lo4a, lo4b;    // b = 4: the 8 magnitudes (levels 8..15), stored sign-magnitude
};
__device__ __forceinline__ uint32_t ld_u32_bytes(const uint8_t *p) { return p[0] | (p[1] << 8) | (p[2] << 16) | ((uint32_t)p[3] << 24); }
__device__ __forceinline__ Pools2 load_pools2(const uint8_t *pl)      // pl: [2][512] planes, flat index 2^b - 1 + k
{
    Pools2 P;
    P.hi2 = ld_u32_bytes(pl + 3);            P.lo2 = ld_u32_bytes(pl + 512 + 3);
    P.hi3a = ld_u32_bytes(pl + 7);           P.hi3b = ld_u32_bytes(pl + 11);
    P.lo3a = ld_u32_bytes(pl + 512 + 7);     P.lo3b = ld_u32_bytes(pl + 512 + 11);
    P.hi4a = ld_u32_bytes(pl + 15 + 8);      P.hi4b = ld_u32_bytes(pl + 15 + 12);
    P.lo4a = ld_u32_bytes(pl + 512 + 15 + 8); P.lo4b = ld_u32_bytes(pl + 512 + 15 + 12);
    return P;
}

// w: the chunk's words of this lane (word j at wp[32 * j]), nw of them in memory.  lut16: [hi | lo << 8] per flat level;
// pair5: [hi_i, hi_j, lo_i, lo_j] for two adjacent 5-bit codes (i = first).
template <int B>
__device__ __forceinline__ void decode_chunk2(const uint32_t *wp, int nw, const Pools2 &P, const uint16_t *lut16,
                                              const uint32_t *pair5, uint32_t (&hi)[8], uint32_t (&lo)[8])
{
    uint32_t w[B];
#pragma unroll
    for (int j = 0; j < B; ++j) w[j] = j < nw ? wp[32 * j] : 0u;
    if constexpr (B == 1) {
#pragma unroll
        for (int Q = 0; Q < 8; ++Q) {                      // slot 4Q+e at bit 8e+7-Q; level 0 = -c, 1 = +c: byte = 0xB8 ^ (bit << 7)
            hi[Q] = ((w[0] << Q) & 0x80808080u) ^ 0xB8B8B8B8u;
            lo[Q] = 0u;
        }
    } else if constexpr (B == 2) {
#pragma unroll
        for (int wi = 0; wi < 2; ++wi)
#pragma unroll
            for (int sub = 0; sub < 2; ++sub) {
                const uint32_t t = (w[wi] >> (2 * sub)) & 0x33333333u;
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {           // quad Q = 2*sub + hf of the word
                    const uint32_t sel = hf ? (t >> 16) : t;
                    hi[wi * 4 + sub * 2 + hf] = prmt(P.hi2, 0u, sel);
                    lo[wi * 4 + sub * 2 + hf] = prmt(P.lo2, 0u, sel);
                }
            }
    } else if constexpr (B == 3 || B == 4) {
        uint32_t t[4];
        t[0] = w[0] & 0x77777777u;
        t[1] = w[1] & 0x77777777u;
        t[2] = w[2] & 0x77777777u;
        t[3] = ((w[0] >> 3) & 0x11111111u) | ((w[1] >> 2) & 0x22222222u) | ((w[2] >> 1) & 0x44444444u);
        const uint32_t Ha = B == 3 ? P.hi3a : P.hi4a, Hb = B == 3 ? P.hi3b : P.hi4b;
        const uint32_t La = B == 3 ? P.lo3a : P.lo4a, Lb = B == 3 ? P.lo3b : P.lo4b;
#pragma unroll
        for (int wi = 0; wi < 4; ++wi)
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const uint32_t sel = hf ? (t[wi] >> 16) : t[wi];
                hi[wi * 2 + hf] = prmt(Ha, Hb, sel);
                lo[wi * 2 + hf] = prmt(La, Lb, sel);
            }
        if constexpr (B == 4) {
            // sign word sits after the magnitude words actually stored: index min(3, ceil(r/8)) = nw - 1
            const uint32_t ws = wp[32 * (nw - 1)];
#pragma unroll
            for (int Q = 0; Q < 8; ++Q) {                  // sign of slot 4Q+e: bit 8e+7-Q; negative level = both planes negated
                const uint32_t sg = (ws << Q) & 0x80808080u;
                hi[Q] ^= sg;
                lo[Q] ^= sg;
            }
        }
    } else {
        auto field = [&](int o, int nbits) -> uint32_t {   // (stream >> o) & (2^nbits - 1)
            const int wi = o >> 5, sh = o & 31;
            uint32_t x;
            if (sh + nbits <= 32) x = w[wi] >> sh;
            else x = __funnelshift_r(w[wi], w[wi + 1 < B ? wi + 1 : wi], sh);
            return x & ((1u << nbits) - 1);
        };
        if constexpr (B == 5) {
#pragma unroll
            for (int Q = 0; Q < 8; ++Q) {
                const uint32_t x = pair5[field(20 * Q, 10)], y = pair5[field(20 * Q + 10, 10)];
                hi[Q] = prmt(x, y, 0x5410);
                lo[Q] = prmt(x, y, 0x7632);
            }
        } else {
            const uint16_t *T = lut16 + ((1 << B) - 1);
#pragma unroll
            for (int Q = 0; Q < 8; ++Q) {
                const uint32_t v0 = T[field(B * (4 * Q), B)], v1 = T[field(B * (4 * Q + 1), B)];
                const uint32_t v2 = T[field(B * (4 * Q + 2), B)], v3 = T[field(B * (4 * Q + 3), B)];
                const uint32_t x = prmt(v0, v1, 0x5140), y = prmt(v2, v3, 0x5140);      // [h0 h1 l0 l1], [h2 h3 l2 l3]
                hi[Q] = prmt(x, y, 0x5410);
                lo[Q] = prmt(x, y, 0x7632);
            }
        }
    }
}

__device__ __forceinline__ void decode_chunk2_any(int b, const uint32_t *wp, int nw, const Pools2 &P, const uint16_t *lut16,
                                                  const uint32_t *pair5, uint32_t (&hi)[8], uint32_t (&lo)[8])
{
    switch (b) {
    case 1: decode_chunk2<1>(wp, nw, P, lut16, pair5, hi, lo); break;
    case 2: decode_chunk2<2>(wp, nw, P, lut16, pair5, hi, lo); break;
    case 3: decode_chunk2<3>(wp, nw, P, lut16, pair5, hi, lo); break;
    case 4: decode_chunk2<4>(wp, nw, P, lut16, pair5, hi, lo); break;
    case 5: decode_chunk2<5>(wp, nw, P, lut16, pair5, hi, lo); break;
    case 6: decode_chunk2<6>(wp, nw, P, lut16, pair5, hi, lo); break;
    case 7: decode_chunk2<7>(wp, nw, P, lut16, pair5, hi, lo); break;
    default: decode_chunk2<8>(wp, nw, P, lut16, pair5, hi, lo); break;
    }
}

__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc2_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc2_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void bar_consumers() { asm volatile("bar.sync 1, %0;" :: "n"(kD2Consumers) : "memory"); }
__device__ __forceinline__ void bar_softmax() { asm volatile("bar.sync 2, 128;" ::: "memory"); }
__device__ __forceinline__ float redux_max(float v)
{
    float r;
    asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
}
// D[128 x 8] (+)= A[128 x 32 e4m3, tensor memory] . B[8 x 32 e4m3, shared memory, K-major SWIZZLE_128B]^T
__device__ __forceinline__ void umma_q8(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_saddr, uint32_t accumulate)
{
    // instruction descriptor: D f32 (1 << 4); A, B e4m3 (0); K-major; N >> 3 = 1 in [17,23); M >> 4 = 8 in [24,29)
    constexpr uint32_t idesc = (1u << 4) | (1u << 17) | (8u << 24);
    const uint64_t db = (uint64_t)((b_saddr & 0x3FFFF) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
                        ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "r"(a_tmem), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit2(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}

// barrier indices (after the ring's full / empty pairs); [2] = double-buffered, indexed by the use's buffer
enum { B2_AK_READY = 0, B2_AK_FREE = 2, B2_S_READY = 4, B2_S_FREE = 6, B2_AV_READY = 8, B2_AV_FREE = 10, B2_P_READY = 12,
       B2_P_FREE = 14, B2_QIMG = 16, B2_COUNT = 17 };

// D[128 x 8] (+)= A . B with the B descriptor given as (constant high part | start address >> 4)
__device__ __forceinline__ void umma_q8d(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t accumulate)
{
    constexpr uint32_t idesc = (1u << 4) | (1u << 17) | (8u << 24);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// D[128 x 24] (+)= A . B, B = three 8-row atoms (SBO = 1024 bytes) of a SWIZZLE_128B image
__device__ __forceinline__ void umma_n24(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t accumulate)
{
    constexpr uint32_t idesc = (1u << 4) | (3u << 17) | (8u << 24);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ uint64_t bdesc_sw128(uint32_t saddr)
{
    return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

#ifndef BGTQ_D2_TIMING
#define BGTQ_D2_TIMING 0
#endif
#if BGTQ_D2_TIMING
#define TWAIT(slot, bar, par) do { long long t0_ = clock64(); mbar_wait(bar, par); twait[slot] += clock64() - t0_; } while (0)
#else
#define TWAIT(slot, bar, par) mbar_wait(bar, par)
#endif

template <bool PAGED>
__global__ void __launch_bounds__(kD2Threads, 1)
decode2_kernel(const Decode2Params P)
{
#if BGTQ_D2_TIMING
    long long twait[6] = {0, 0, 0, 0, 0, 0};
    const long long tstart = clock64();
#endif
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // dynamic (1024-byte aligned by hand: the SWIZZLE_128B pattern is a function of the address):
    // [q' image 10 KB][P' planes 2 x 3 KB][ring: n_stages x stage_bytes]
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char *qimg_s = smem;
    unsigned char *pimg_s = smem + 10 * 1024;
    unsigned char *ring = smem + 16 * 1024;
    __shared__ __align__(8) HeadMeta Ms;
    __shared__ __align__(16) uint8_t planes_s[kPlaneBytes];
    __shared__ __align__(16) uint16_t lut16[512];
    __shared__ __align__(16) uint32_t pair5[1024];
    __shared__ int pre[kMaxBatch + 1];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages + B2_COUNT];
    __shared__ uint32_t tmem_base_s;
    __shared__ float qmax_s[2][4][8];
    __shared__ float lsum_s[4][8];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int quad = warp & 3;
    // roles: 0 K unpack (warps 0-3), 1 softmax (4-7), 2 V unpack (8-11), 4 TMA (12), 3 QK^T issue (13 ..), 5 PV issue (the last two)
    const int role = warp < 12 ? (warp >> 2) : (warp == 12 ? 4 : (warp < 13 + kQkIssuers ? 3 : 5));
    const int issuer = warp < 13 + kQkIssuers ? warp - 13 : warp - 13 - kQkIssuers;
    pdl_trigger();

    for (int i = tid; i < kPlaneBytes; i += kD2Threads) planes_s[i] = __ldg(P.planes + i);
    for (int i = tid; i < 2 * kP2Bytes / 16; i += kD2Threads) reinterpret_cast<uint4 *>(pimg_s)[i] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0) build_prefix(P.seq_len, P.batch, P.n_cap * kTile, pre, P.n_sink, P.n_recent);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" :: "r"(smem_u32(&tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    const uint32_t bar0 = smem_u32(bars);
    auto full_bar = [&](int s) { return bar0 + 8u * s; };
    auto empty_bar = [&](int s) { return bar0 + 8u * (kMaxStages + s); };
    auto xbar = [&](int i) { return bar0 + 8u * (2 * kMaxStages + i); };
    if (tid == 32) {
        for (int s = 0; s < P.n_stages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 12); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(xbar(B2_AK_READY + b), 4);  mbar_init(xbar(B2_AK_FREE + b), kQkIssuers);
            mbar_init(xbar(B2_S_READY + b), kQkIssuers);   mbar_init(xbar(B2_S_FREE + b), 4);
            mbar_init(xbar(B2_AV_READY + b), 4);  mbar_init(xbar(B2_AV_FREE + b), kPvIssuers);
            mbar_init(xbar(B2_P_READY + b), 4);   mbar_init(xbar(B2_P_FREE + b), kPvIssuers);
        }
        mbar_init(xbar(B2_QIMG), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    tc2_fence_before();
    __syncthreads();
    tc2_fence_after();
    for (int i = tid; i < 511; i += kD2Threads) lut16[i] = (uint16_t)(planes_s[i] | (planes_s[512 + i] << 8));
    for (int i = tid; i < 1024; i += kD2Threads) {
        const int a = 31 + (i & 31), b = 31 + (i >> 5);                       // first code = low 5 bits of the 10-bit field
        pair5[i] = planes_s[a] | (planes_s[b] << 8) | (planes_s[512 + a] << 16) | ((uint32_t)planes_s[512 + b] << 24);
    }
    __syncthreads();

    const uint32_t tmem = tmem_base_s;
    const Sched S = make_sched(P.n_layers, P.batch, P.Hkv, pre, gridDim.x, 1);
    const int x_lo = cta_lo(S, blockIdx.x), x_hi = cta_lo(S, blockIdx.x + 1);
    auto tile_src = [&](const TilePos &tp, const HeadMeta &M) -> const uint8_t * {
        if (PAGED)
            return P.cache + P.n_pages * ((int64_t)M.layer_prefix + M.head_prefix) +
                   (int64_t)__ldg(P.pages + (int64_t)tp.b * P.pstride + tp.t) * M.tile_stride;
        return P.cache + P.n_cap * ((int64_t)P.batch * M.layer_prefix + (int64_t)tp.b * M.layer_sum + M.head_prefix) +
               (int64_t)tp.t * M.tile_stride;
    };

    // ================================================================ TMA producer: free-runs over the CTA's tile range
    if (role == 4) {
        if (lane == 0) {
            int it = 0;
            for (int x = x_lo; x < x_hi;) {
                const TilePos tp = locate(x, S, pre);
                const HeadMeta &M = P.metas[tp.l * P.Hkv + tp.h];
                const int seg_end = min(x_hi, tp.pair_start + tp.tiles_b);
                const uint32_t stride = (uint32_t)__ldg(&M.tile_stride);
                const uint8_t *src = tile_src(tp, M);
                const uint8_t *pool = P.cache + P.n_pages * ((int64_t)M.layer_prefix + M.head_prefix);
                const int32_t *prow = P.pages + (int64_t)tp.b * P.pstride;
                for (int t = tp.t; x < seg_end; ++x, ++t, ++it) {
                    const int s = it % P.n_stages;
                    if (it >= P.n_stages) mbar_wait(empty_bar(s), ((it / P.n_stages) - 1) & 1);
                    if (PAGED) src = pool + (int64_t)__ldg(prow + t) * stride;
                    mbar_expect_tx(full_bar(s), stride);
                    bulk_g2s(smem_u32(ring + (size_t)s * P.stage_bytes), src, stride, full_bar(s));
                    src += stride;
                }
            }
        }
        // the producer warp leaves; the copies it issued complete on their mbarriers (consumers wait for all of them)
        return;
    }

    // Every wait below derives its parity from the tile counter `it` (tiles consumed by this CTA so far): a resource with
    // nb buffers is used for the (it / nb)-th time by tile it, in buffer it % nb.
    const Pools2 pools = load_pools2(planes_s);
    const int nbk = P.ak_bufs;
    int it = 0, seg = 0;
    const uint32_t lane_base = (uint32_t)(32 * quad) << 16;
    auto ak_col = [&](int buf, int plane, int ch) { return kColAK + (nbk == 2 ? buf * 96 + plane * 48 : plane * 96) + 8 * ch; };
    auto av_col = [&](int buf, int plane, int c) { return kColAV + buf * 64 + plane * 32 + 8 * c; };

    for (int x = x_lo; x < x_hi; ++seg) {
        // ---------------- segment = the part of one (layer, sequence, kv head) inside this CTA's range
        const TilePos tp = locate(x, S, pre);
        const int seg_end = min(x_hi, tp.pair_start + tp.tiles_b);
        bar_consumers();                                // every consumer is done with the previous segment's metadata / q' image
        {
            const uint32_t *msrc = reinterpret_cast<const uint32_t *>(P.metas + tp.l * P.Hkv + tp.h);
            if (tid < (int)(sizeof(HeadMeta) / 4)) reinterpret_cast<uint32_t *>(&Ms)[tid] = __ldg(msrc + tid);
        }
        if (role == 3 && issuer == 0 && lane == 0) {    // q' image of this pair (written by qfold2_kernel)
            pdl_wait();
            mbar_expect_tx(xbar(B2_QIMG), kQ2Stride);
            bulk_g2s(smem_u32(qimg_s), P.qimg + (size_t)tp.pair * kQ2Stride, kQ2Stride, xbar(B2_QIMG));
        }
        bar_consumers();
        const HeadMeta &M = Ms;
        const int n_chunks = M.n_ksteps, n_groups = M.n_groups, b_v = M.b_v;
        int64_t slen = P.seq_len[tp.b];
        slen = slen > P.n_cap * kTile ? P.n_cap * kTile : slen;
        slen = packed_len(slen, P.n_sink, P.n_recent);
        const int n_tiles_seg = seg_end - x;
        x = seg_end;

        if (role == 0) {
            // ======================================================== K unpack: thread = token row `quad*32 + lane`
            const int kq4 = M.kcode_bytes >> 4;                          // words of one quadrant's K-code section
            for (int j = 0; j < n_tiles_seg; ++j, ++it) {
                const int s = it % P.n_stages;
                TWAIT(0, full_bar(s), (it / P.n_stages) & 1);
                const uint32_t *kc = reinterpret_cast<const uint32_t *>(ring + (size_t)s * P.stage_bytes) + quad * kq4 + lane;
                const int buf = it % nbk, use = it / nbk;
                bool waited = use == 0;
#pragma unroll 1
                for (int ch = 0; ch < n_chunks; ++ch) {
                    const Chunk2 C2 = M.chunks[ch];
                    uint32_t hi[8], lo[8];
                    decode_chunk2_any(C2.b, kc + (C2.off >> 2), C2.nw, pools, lut16, pair5, hi, lo);
                    if (!waited) { TWAIT(1, xbar(B2_AK_FREE + buf), (use - 1) & 1); tc2_fence_after(); waited = true; }
                    tmem_st8(tmem + lane_base + ak_col(buf, 0, ch), hi);
                    if (C2.b > 1) tmem_st8(tmem + lane_base + ak_col(buf, 1, ch), lo);
                }
#if BGTQ_D2_TIMING
                long long tq0 = clock64();
#endif
                tmem_wait_st();
#if BGTQ_D2_TIMING
                twait[3] += clock64() - tq0;
#endif
                tc2_fence_before();
                __syncwarp();
                if (lane == 0) { mbar_arrive(xbar(B2_AK_READY + buf)); mbar_arrive(empty_bar(s)); }
            }
        } else if (role == 2) {
            // ======================================================== V unpack: thread = dimension row `quad*32 + lane`
            for (int j = 0; j < n_tiles_seg; ++j, ++it) {
                const int s = it % P.n_stages;
                TWAIT(0, full_bar(s), (it / P.n_stages) & 1);
                const uint32_t *vc = reinterpret_cast<const uint32_t *>(ring + (size_t)s * P.stage_bytes + M.vcode_off) + quad * 4 * b_v * 32 + lane;
                const int buf = it & 1, use = it >> 1;
                bool waited = use == 0;
#pragma unroll 1
                for (int c = 0; c < 4; ++c) {
                    uint32_t hi[8], lo[8];
                    decode_chunk2_any(b_v, vc + c * b_v * 32, b_v, pools, lut16, pair5, hi, lo);
                    if (!waited) { TWAIT(1, xbar(B2_AV_FREE + buf), (use - 1) & 1); tc2_fence_after(); waited = true; }
                    tmem_st8(tmem + lane_base + av_col(buf, 0, c), hi);
                    if (b_v > 1) tmem_st8(tmem + lane_base + av_col(buf, 1, c), lo);
                }
                tmem_wait_st();
                tc2_fence_before();
                __syncwarp();
                if (lane == 0) { mbar_arrive(xbar(B2_AV_READY + buf)); mbar_arrive(empty_bar(s)); }
            }
        } else if (role == 3) {
            // ======================================================== QK^T issue: S_g = A_K . q' ; issuer i owns the groups g = i (mod kQkIssuers)
            if (lane == 0) {
                mbar_wait(xbar(B2_QIMG), seg & 1);
                const uint64_t qd = bdesc_sw128(smem_u32(qimg_s));
                for (int j = 0; j < n_tiles_seg; ++j, ++it) {
                    const int bufk = it % nbk, sb = it & 1;
                    TWAIT(1, xbar(B2_AK_READY + bufk), (it / nbk) & 1);
                    if (it >= 2) TWAIT(2, xbar(B2_S_FREE + sb), ((it >> 1) - 1) & 1);
                    tc2_fence_after();
                    for (int ch = 0; ch < n_chunks; ++ch) {
                        const Chunk2 C2 = M.chunks[ch];
                        const int g = C2.flags >> 4;
                        if (g % kQkIssuers != issuer) continue;
                        const uint32_t d = tmem + kColS + 64 * sb + 8 * g;
                        const uint32_t ahi = tmem + ak_col(bufk, 0, ch), alo = tmem + ak_col(bufk, 1, ch);
                        const int sl = 3 * ch;
                        auto bq = [&](int p) { return qd + (uint64_t)((((sl + p) >> 2) * 1024 + ((sl + p) & 3) * 32) >> 4); };
                        umma_q8d(d, ahi, bq(0), (C2.flags & 1) ? 0u : 1u);
                        umma_q8d(d, ahi, bq(1), 1u);
                        umma_q8d(d, ahi, bq(2), 1u);
                        if (C2.b > 1) { umma_q8d(d, alo, bq(0), 1u); umma_q8d(d, alo, bq(1), 1u); }
                    }
                    umma_commit2(xbar(B2_S_READY + sb));
                    umma_commit2(xbar(B2_AK_FREE + bufk));
                }
            } else it += n_tiles_seg;
            __syncwarp();
        } else if (role == 5) {
            // ======================================================== PV issue: O[128 dims x (3 planes x 8 heads)] += A_V . P'; issuer 0 = hi plane of V, 1 = lo plane
            if (lane == 0) {
                const uint64_t pd = bdesc_sw128(smem_u32(pimg_s));
                for (int j = 0; j < n_tiles_seg; ++j, ++it) {
                    const int b = it & 1;
                    TWAIT(1, xbar(B2_AV_READY + b), (it >> 1) & 1);
                    TWAIT(2, xbar(B2_P_READY + b), (it >> 1) & 1);
                    tc2_fence_after();
                    if (issuer == 0 || b_v > 1)
                        for (int c = 0; c < 4; ++c)        // (O was zeroed by the softmax warps before the first P' of the segment)
                            umma_n24(tmem + kColO, tmem + av_col(b, issuer, c), pd + (uint64_t)((b * kP2Bytes + 32 * c) >> 4), 1u);
                    umma_commit2(xbar(B2_AV_FREE + b));
                    umma_commit2(xbar(B2_P_FREE + b));
                }
            } else it += n_tiles_seg;
            __syncwarp();
        } else {
            // ======================================================== softmax: thread = token row `quad*32 + lane`
            mbar_wait(xbar(B2_QIMG), seg & 1);                      // sigma_n arrives with the q' image
            float sig[8];
#pragma unroll
            for (int n = 0; n < 8; ++n) sig[n] = reinterpret_cast<const float *>(qimg_s + kQ2ImageBytes)[n];
            float R[8], lacc[8];
#pragma unroll
            for (int n = 0; n < 8; ++n) { R[n] = -INFINITY; lacc[n] = 0.f; }
            const int row = quad * 32 + lane;
            {   // O = 0: both PV issuers only ever accumulate.  The previous segment's record has been read (its PV was complete).
                const uint32_t z[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
                tmem_st8(tmem + lane_base + kColO + 0, z);
                tmem_st8(tmem + lane_base + kColO + 8, z);
                tmem_st8(tmem + lane_base + kColO + 16, z);
                tmem_wait_st();
                tc2_fence_before();
            }
            for (int j = 0, t = tp.t; j < n_tiles_seg; ++j, ++t, ++it) {
                const int s = it % P.n_stages, sb = it & 1;
                TWAIT(0, full_bar(s), (it / P.n_stages) & 1);
                const unsigned char *tile = ring + (size_t)s * P.stage_bytes;
                // norms of this token: K groups, V
                float nk[kMaxGroups];
#pragma unroll
                for (int g = 0; g < kMaxGroups; ++g)
                    nk[g] = g < n_groups ? __half2float(reinterpret_cast<const __half *>(tile + M.knorm_off + 256 * g)[row]) : 0.f;
                const float hv = __half2float(reinterpret_cast<const __half *>(tile + M.vnorm_off)[row]);
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_bar(s));
                const float hve = hv > 0.f ? hv : 5.9604645e-8f;      // 2^-24 stands in for a zero norm in the denominator path only
                const float lgh = __log2f(hve), rh = __frcp_rn(hve);
                const int n_valid = (int)min((int64_t)kTile, slen - (int64_t)t * kTile);
                const int n_low = t == 0 ? P.n_sink : 0;
                const bool live = row < n_valid && row >= n_low;
                // ---- logits: all group accumulators are requested, then one wait
                TWAIT(1, xbar(B2_S_READY + sb), (it >> 1) & 1);
                tc2_fence_after();
                float lg[8];
#pragma unroll
                for (int n = 0; n < 8; ++n) lg[n] = 0.f;
#pragma unroll
                for (int g0 = 0; g0 < kMaxGroups; g0 += 4) {        // four groups per round trip to tensor memory
                    if (g0 < n_groups) {
                        uint32_t sv[4][8];
#pragma unroll
                        for (int g = 0; g < 4; ++g)
                            if (g0 + g < n_groups) tmem_ld8(tmem + lane_base + kColS + 64 * sb + 8 * (g0 + g), sv[g]);
                        tmem_wait_ld();
#pragma unroll
                        for (int g = 0; g < 4; ++g)
                            if (g0 + g < n_groups) {
#pragma unroll
                                for (int n = 0; n < 8; ++n) lg[n] = fmaf(nk[g0 + g], __uint_as_float(sv[g][n]), lg[n]);
                            }
                    }
                }
                tc2_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(xbar(B2_S_FREE + sb));
#pragma unroll
                for (int n = 0; n < 8; ++n) lg[n] = live ? fmaf(lg[n], sig[n], lgh) : -INFINITY;
                // ---- reference update (CTA-wide, per head): quadrant maxima meet in shared memory (double-buffered by tile parity)
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const float m = redux_max(lg[n]);
                    if (lane == n) qmax_s[sb][quad][n] = m;
                }
                bar_softmax();
                float alpha[8];
                bool any = false;
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const float tm = fmaxf(fmaxf(qmax_s[sb][0][n], qmax_s[sb][1][n]), fmaxf(qmax_s[sb][2][n], qmax_s[sb][3][n]));
                    alpha[n] = 1.f;
                    if (tm > R[n] + kRefLimit) {
                        const float Rn = tm - kRefHeadroom;
                        alpha[n] = fast_exp2(R[n] - Rn);            // 0 for the first reference
                        R[n] = Rn;
                        any = any || (n < P.G && j > 0);
                    }
                }
                if (any) {
                    // rare: rescale the accumulators in tensor memory.  The PV of tile it - 1 must be complete.
                    mbar_wait(xbar(B2_P_FREE + ((it - 1) & 1)), ((it - 1) >> 1) & 1);
                    tc2_fence_after();
#pragma unroll
                    for (int p = 0; p < 3; ++p) {
                        uint32_t ov[8];
                        tmem_ld8(tmem + lane_base + kColO + 8 * p, ov);
                        tmem_wait_ld();
#pragma unroll
                        for (int n = 0; n < 8; ++n) ov[n] = __float_as_uint(__uint_as_float(ov[n]) * alpha[n]);
                        tmem_st8(tmem + lane_base + kColO + 8 * p, ov);
                    }
                    tmem_wait_st();
                    tc2_fence_before();
                    bar_softmax();
                }
                // ---- weights: P' = 2^(lg - R) in three e4m3 planes of ratio 2^-4; l += P' / h^V
                uint32_t p1[2] = {0u, 0u}, p2[2] = {0u, 0u}, p3[2] = {0u, 0u};
#pragma unroll
                for (int n = 0; n < 8; n += 2) {
                    const float x0 = fast_exp2(lg[n] - R[n]), x1 = fast_exp2(lg[n + 1] - R[n + 1]);
                    lacc[n] = fmaf(lacc[n], alpha[n], x0 * rh);
                    lacc[n + 1] = fmaf(lacc[n + 1], alpha[n + 1], x1 * rh);
                    const float y0 = hv > 0.f ? x0 : 0.f, y1 = hv > 0.f ? x1 : 0.f;
                    const uint32_t a = cvt_e4m3x2(y0, y1);
                    const float2 af = e4m3x2_to_f32(a);
                    // (a rounding error is at most 2^-4 of the value, so 16 x the residual stays inside the e4m3 range)
                    const float r0 = (y0 - af.x) * 16.f, r1 = (y1 - af.y) * 16.f;
                    const uint32_t b = cvt_e4m3x2(r0, r1);
                    const float2 bf = e4m3x2_to_f32(b);
                    const uint32_t c = cvt_e4m3x2((r0 - bf.x) * 16.f, (r1 - bf.y) * 16.f);
                    p1[n >> 2] |= a << (8 * (n & 3));
                    p2[n >> 2] |= b << (8 * (n & 3));
                    p3[n >> 2] |= c << (8 * (n & 3));
                }
                // ---- planes -> shared memory (B operand of PV: row = head, K = token); buffer it & 1
                if (it >= 2) TWAIT(2, xbar(B2_P_FREE + sb), ((it >> 1) - 1) & 1);
                unsigned char *pi = pimg_s + sb * kP2Bytes;
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    pi[sw128_off(0 + quad, n, lane)] = (uint8_t)(p1[n >> 2] >> (8 * (n & 3)));     // atom = plane, 32-byte K slice = token quarter
                    pi[sw128_off(4 + quad, n, lane)] = (uint8_t)(p2[n >> 2] >> (8 * (n & 3)));
                    pi[sw128_off(8 + quad, n, lane)] = (uint8_t)(p3[n >> 2] >> (8 * (n & 3)));
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(xbar(B2_P_READY + sb));
            }
            // ---------------- segment end: one partial record (R, l, acc[128]) per head; this warp owns dims quad*32 + lane
            {
                mbar_wait(xbar(B2_P_FREE + ((it - 1) & 1)), ((it - 1) >> 1) & 1);     // PV of the last tile complete
                tc2_fence_after();
                float o[8];
                {
                    uint32_t o1[8], o2[8], o3[8];
                    tmem_ld8(tmem + lane_base + kColO + 0, o1);
                    tmem_ld8(tmem + lane_base + kColO + 8, o2);
                    tmem_ld8(tmem + lane_base + kColO + 16, o3);
                    tmem_wait_ld();
#pragma unroll
                    for (int n = 0; n < 8; ++n)
                        o[n] = (__uint_as_float(o1[n]) + __uint_as_float(o2[n]) * 0.0625f + __uint_as_float(o3[n]) * 0.00390625f) * P.inv_kappa_v;
                }
                tc2_fence_before();
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    float v = lacc[n];
#pragma unroll
                    for (int sft = 16; sft; sft >>= 1) v += __shfl_xor_sync(0xffffffffu, v, sft);
                    if (lane == n) lsum_s[quad][n] = v;
                }
                bar_softmax();
                float *rec = P.partials + (size_t)(blockIdx.x + tp.pair) * kPartialFloats;
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    if (n < P.G) {
                        rec[n * 130 + 2 + row] = o[n];
                        if (row == n) {
                            rec[n * 130] = R[n];
                            rec[n * 130 + 1] = (lsum_s[0][n] + lsum_s[1][n]) + (lsum_s[2][n] + lsum_s[3][n]);
                        }
                    }
                }
                bar_softmax();
            }
        }
    }
#if BGTQ_D2_TIMING
    if (blockIdx.x == 3 && lane == 0 && (quad == 0 || role >= 3))
        printf("role %d warp %2d: total %lld  wait full %lld  wait[1] %lld  wait[2] %lld  wait_st %lld tiles %d\n", role, warp, clock64() - tstart,
               twait[0], twait[1], twait[2], twait[3], it);
#endif
    tc2_fence_before();
    bar_consumers();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tmem) : "memory");
}

// ---------------------------------------------------------------- host side
size_t decode2_ws_bytes(const bgtq_layout *lay, int batch, int n_layers)
{
    const size_t pairs = (size_t)n_layers * batch * lay->n_kv_heads;
    const size_t slots = (size_t)lay->sm_count + 2 * pairs;          // one record per (CTA, pair) + one window record per pair
    return pairs * kQ2Stride + slots * kPartialFloats * sizeof(float);
}

int launch_decode2(const bgtq_layout *lay, int layer0, int n_layers, const void *cache, const void *q,
                   const int32_t *seq_len, int batch, int64_t max_tokens, float scale, void *out,
                   void *ws, size_t, const PageMap *pm, cudaStream_t st, const Window *win)
{
    const int n_sink = win ? win->n_sink : 0, n_recent = win ? win->n_recent : 0;
    if (batch > kMaxBatch) { set_error("bgtq_decode_attention: batch > 256"); return BGTQ_EINVAL; }
    const int Hkv = lay->n_kv_heads, Hq = lay->n_q_heads, G = Hq / Hkv;
    const int64_t n_cap = (max_tokens + kTile - 1) / kTile;
    if ((double)n_layers * batch * Hkv * (double)n_cap >= 2.0e9) { set_error("bgtq_decode_attention: too many tiles for one call"); return BGTQ_EINVAL; }
    const int pairs = n_layers * batch * Hkv;
    uint8_t *qimg = reinterpret_cast<uint8_t *>(ws);
    float *partials = reinterpret_cast<float *>(qimg + (size_t)pairs * kQ2Stride);
    const HeadMeta *metas = lay->d_meta + (size_t)layer0 * Hkv;
    const bool prof = profile_decode_on();
    const int grid = lay->sm_count;
    const int win_slot = win ? grid + pairs : -1;
    const float sl2e = scale * 1.4426950408889634f;
    static float *d_kappa = nullptr;                 // kappa[0..8] (the same for every layout: it depends on the codebooks only)
    if (!d_kappa) {
        CUDA_TRY(cudaMalloc(&d_kappa, 9 * sizeof(float)));
        CUDA_TRY(cudaMemcpy(d_kappa, lay->kappa, 9 * sizeof(float), cudaMemcpyHostToDevice));
    }
    if (win) {
        if (int rc = launch_window(win->k, win->v, q, seq_len, lay->d_rot_t + rot_offset(kDh), partials, pairs, batch, Hkv, G, n_cap,
                                   n_sink, n_recent, sl2e, win_slot, st)) return rc;
    }
    {
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = (win && !prof) ? 1 : 0;
        cfg.gridDim = dim3(pairs * G); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 0; cfg.stream = st;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, qfold2_kernel, metas, (const float *)lay->d_rot_t, (const __nv_bfloat16 *)q, batch, Hkv, Hq, sl2e,
                           (const float *)d_kappa, qimg);
        count_launch();
        CUDA_TRY(cudaGetLastError());
    }
    Decode2Params P;
    P.metas = metas; P.cache = (const uint8_t *)cache; P.qimg = qimg; P.seq_len = seq_len; P.planes = lay->d_planes;
    P.partials = partials; P.n_cap = n_cap; P.n_layers = n_layers; P.batch = batch; P.Hkv = Hkv; P.G = G;
    P.stage_bytes = (lay->max_stride + 127) / 128 * 128;
    const int static_smem = 12 * 1024;                               // upper bound of the kernel's static shared memory
    const int avail = 227 * 1024 - static_smem - 17 * 1024;           // 16 KB of operand images + 1 KB alignment slack
    P.n_stages = avail / P.stage_bytes;
    if (P.n_stages > kMaxStages) P.n_stages = kMaxStages;
    if (P.n_stages < 2) { set_error("bgtq_decode_attention: tile does not fit shared memory"); return BGTQ_EINVAL; }
    P.inv_kappa_v = 1.0f / lay->kappa[lay->b_v];
    P.ak_bufs = lay->max_chunks <= 6 ? 2 : 1;
    P.pages = pm ? pm->table : nullptr; P.pstride = pm ? pm->table_stride : 0; P.n_pages = pm ? pm->n_pages : 0;
    P.n_sink = n_sink; P.n_recent = n_recent;
    const size_t smem = 17 * 1024 + (size_t)P.n_stages * P.stage_bytes;
    if (first_use_on_device(4)) {
        CUDA_TRY(cudaFuncSetAttribute(decode2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - static_smem));
        CUDA_TRY(cudaFuncSetAttribute(decode2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - static_smem));
    }
    if (int rc = profile_decode_begin(st)) return rc;
    {
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = prof ? 0 : 1;
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kD2Threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cfg.attrs = at; cfg.numAttrs = 1;
        if (pm) cudaLaunchKernelEx(&cfg, decode2_kernel<true>, P);
        else cudaLaunchKernelEx(&cfg, decode2_kernel<false>, P);
        cudaError_t le = cudaPeekAtLastError();
        if (le != cudaSuccess) {
            cudaFuncAttributes fa;
            cudaFuncGetAttributes(&fa, decode2_kernel<false>);
            set_error(std::string("decode2 launch: ") + cudaGetErrorString(le) + " regs=" + std::to_string(fa.numRegs) + " static=" +
                      std::to_string(fa.sharedSizeBytes) + " dyn=" + std::to_string(smem));
            cudaGetLastError();
            return BGTQ_ECUDA;
        }
        count_launch();
    }
    if (int rc = profile_decode_end(st)) return rc;
    return launch_combine(partials, seq_len, lay->d_rot + rot_offset(kDh), n_layers, batch, Hkv, G, n_cap, grid, 1, out, n_sink,
                          n_recent, win_slot, !prof, st);
}

}  // namespace bgtq
