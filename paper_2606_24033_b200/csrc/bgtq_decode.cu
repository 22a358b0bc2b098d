// bgtq_decode.cu -- split-KV decode attention over the packed cache and the exact
// log-sum-exp combine + V de-rotation (a6).  PAPER.md:114, 120.  Hand-written for sm_100a.
//
// Algebra: the TQ-MSE rotation is folded into the query once per call
//   q'_g = Pi^(m_g) q_g * (scale*log2(e)/sqrt(m_g))          (prologue kernel)
// so that  log2e*logit_t = sum_g h_{t,g} * sum_j q'_{g,j} C_{b_g}[idx_{t,g,j}]  -- no key is ever
// de-rotated and no fp16 K/V tile exists outside registers.  V is accumulated in the rotated
// domain and de-rotated once per query head after the cross-split merge.
//
// Mapping: one WARP owns one 128-token tile at a time.  The tile is one contiguous range of the
// cache and is staged into the warp's private shared-memory buffer by two TMA bulk copies
// (cp.async.bulk + mbarrier): [K codes|K norms] and [V norms|V codes]; the K half of the next
// tile is requested as soon as QK^T of the current one is done, the V half after PV, so the copy
// engine runs one half-tile ahead of the math of every warp.  Codes are laid out in mma.sync
// fragment order: tokens are the M dimension of QK^T (A = unpacked codes, fp16
// exact; B = q' for the <= 8 query heads of the GQA group), dims are the M dimension of PV.
// Work is split over ALL warps of the grid in equal contiguous ranges of the global tile list
// [layer][sequence][kv head][tile] (flash-decoding along the key axis); a warp writes
// one partial (max, sum, acc[128]) per (pair, warp) it touches.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <cstdlib>
#include <utility>
#include <vector>

#include "bgtq_internal.h"
#include "bgtq_device.cuh"

namespace bgtq {

static_assert(sizeof(HeadMeta) % 4 == 0 && sizeof(HeadMeta) <= 128 * 4, "qfold_kernel copies HeadMeta with one word per thread");

#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

#ifndef BGTQ_NORM_IN_OPERAND
#define BGTQ_NORM_IN_OPERAND 0   // 1: fold K group norms into the fp16 A operand (measured: no faster, less exact); 0: scale fp32 accumulators
#endif
#ifndef BGTQ_TIMING
#define BGTQ_TIMING 0
#endif
#ifndef BGTQ_NO_P5
#define BGTQ_NO_P5 0
#endif
constexpr int kQfHalves = kMaxKSteps * 8 * 16;      // fp16 q' fragments per (layer, seq, kv head)

// Optional: shifts issued to the FMA pipe (IMAD) instead of the ALU pipe (tuning switches)
__device__ __forceinline__ uint32_t shl_k(uint32_t x, int k)
{
#ifdef BGTQ_SHL_FMA
    uint32_t r;
    asm("mul.lo.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(1u << k));
    return r;
#else
    return x << k;
#endif
}
__device__ __forceinline__ uint32_t shr16(uint32_t x)
{
#ifdef BGTQ_SHR16_FMA
    uint32_t r;
    asm("mul.hi.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(0x10000u));
    return r;
#elif defined(BGTQ_SHR16_PRMT)
    return prmt(x, 0u, 0x4432);
#else
    return x >> 16;
#endif
}

// ---------------------------------------------------------------- unit decoders
// A unit = B words per lane holding 32 slots.  Output: 16 half2 registers,
// h[j] = (slot 2j, slot 2j+1) as fp16 codebook values (exact: the codebook is fp16).
// pools[]: byte planes of the small codebooks for PRMT lookups, built once per CTA:
//   [0]      b=1: (0x8000 | +c) in both halves
//   [1],[2]  b=2: low bytes / high bytes of levels 0..3
//   [3..6]   b=3: low bytes of levels 0..3, 4..7; high bytes of levels 0..3, 4..7
//   [7..10]  b=4: same for the 8 magnitudes C_4[8..15] (codes are stored sign-magnitude)
// lut: fp16 bits of the flat codebook table in shared memory (C_b at 2^b - 1), for b >= 5.
template <int B, bool P5 = true>
__device__ __forceinline__ void decode_unit(const uint32_t (&w)[B], const uint32_t *pools,
                                            const uint16_t *lut, uint32_t (&h)[16])
{
    if constexpr (B == 1) {
        const uint32_t mag = pools[0];
#pragma unroll
        for (int j = 0; j < 16; ++j) h[j] = ((j ? shl_k(w[0], j) : w[0]) & 0x80008000u) ^ mag;
    } else if constexpr (B == 2) {
        const uint32_t LO = pools[1], HI = pools[2];
#pragma unroll
        for (int wi = 0; wi < 2; ++wi)
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const uint32_t t = (w[wi] >> (2 * hf)) & 0x33333333u;
#pragma unroll
                for (int ql = 0; ql < 2; ++ql) {
                    const uint32_t sel = ql ? shr16(t) : t;
                    const uint32_t lo4 = prmt(LO, 0, sel), hi4 = prmt(HI, 0, sel);
                    const int Q = hf * 2 + ql;
                    h[wi * 8 + 2 * Q] = prmt(lo4, hi4, 0x5140);
                    h[wi * 8 + 2 * Q + 1] = prmt(lo4, hi4, 0x7362);
                }
            }
    } else if constexpr (B == 3 || B == 4) {
        const int pb = B == 3 ? 3 : 7;
        const uint32_t LOa = pools[pb], LOb = pools[pb + 1], HIa = pools[pb + 2], HIb = pools[pb + 3];
        uint32_t t[4];
        t[0] = w[0] & 0x77777777u;
        t[1] = w[1] & 0x77777777u;
        t[2] = w[2] & 0x77777777u;
        t[3] = ((w[0] >> 3) & 0x11111111u) | ((w[1] >> 2) & 0x22222222u) | ((w[2] >> 1) & 0x44444444u);
#pragma unroll
        for (int wi = 0; wi < 4; ++wi)
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const uint32_t sel = hf ? shr16(t[wi]) : t[wi];
                uint32_t lo4 = prmt(LOa, LOb, sel), hi4 = prmt(HIa, HIb, sel);
                if constexpr (B == 4) hi4 ^= ((2 * wi + hf) ? shl_k(w[3], 2 * wi + hf) : w[3]) & 0x80808080u;   // sign of slot 4Q+e: bit 8e+7-Q
                h[wi * 4 + 2 * hf] = prmt(lo4, hi4, 0x5140);
                h[wi * 4 + 2 * hf + 1] = prmt(lo4, hi4, 0x7362);
            }
    } else {
        // byte offset of the table entry straight from the bit stream: one shift (funnel when the
        // field straddles two words) + one mask, then LDS [offset + constant table address].
        auto field_off = [&](int o, int nbits, int scale_log2) -> uint32_t {   // ((stream >> o) & (2^nbits-1)) << scale_log2
            const int wi = o >> 5, sh = (o & 31) - scale_log2;
            uint32_t x;
            if (sh < 0) x = w[wi] << (-sh);
            else if (sh + scale_log2 + nbits <= 32) x = w[wi] >> sh;
            else x = __funnelshift_r(w[wi], w[wi + 1 < B ? wi + 1 : wi], sh);
            return x & (((1u << nbits) - 1) << scale_log2);
        };
        if constexpr (B == 5 && P5) {      // pair table: 1024 half2 entries indexed by two adjacent 5-bit codes
            const char *T2 = reinterpret_cast<const char *>(lut + 512);
#pragma unroll
            for (int j = 0; j < 16; ++j) h[j] = *reinterpret_cast<const uint32_t *>(T2 + field_off(10 * j, 10, 2));
        } else {
            const char *T = reinterpret_cast<const char *>(lut + ((1 << B) - 1));
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const uint32_t v0 = *reinterpret_cast<const uint16_t *>(T + field_off(B * (2 * j), B, 1));
                const uint32_t v1 = *reinterpret_cast<const uint16_t *>(T + field_off(B * (2 * j + 1), B, 1));
                h[j] = prmt(v0, v1, 0x5410);
            }
        }
    }
}

constexpr int kLutHalves = 512 + 2048;     // flat fp16 codebooks (C_b at 2^b-1) + the 5-bit pair table
__device__ __forceinline__ void build_lut(const uint16_t *cb16_global, uint16_t *lut, int tid, int nthreads, bool pair5 = true)
{
    for (int i = tid; i < 512; i += nthreads) lut[i] = cb16_global[i < 511 ? i : 510];
    uint32_t *pair = reinterpret_cast<uint32_t *>(lut + 512);
    for (int i = tid; i < (pair5 ? 1024 : 0); i += nthreads)
        pair[i] = (uint32_t)cb16_global[31 + (i & 31)] | ((uint32_t)cb16_global[31 + (i >> 5)] << 16);
}

__device__ __forceinline__ void build_pools(const uint16_t *cb16, uint32_t *pools)
{
    // cb16: flat fp16 table in shared memory; one thread fills all pools (tiny)
    pools[0] = (0x8000u | cb16[1 + 1]) * 0x10001u;
    auto plane = [&](int base, int hi) {
        uint32_t r = 0;
        for (int k = 0; k < 4; ++k) r |= (uint32_t)((cb16[base + k] >> (hi ? 8 : 0)) & 0xFF) << (8 * k);
        return r;
    };
    pools[1] = plane(3, 0);  pools[2] = plane(3, 1);
    pools[3] = plane(7, 0);  pools[4] = plane(11, 0); pools[5] = plane(7, 1);  pools[6] = plane(11, 1);
    pools[7] = plane(15 + 8, 0); pools[8] = plane(15 + 12, 0); pools[9] = plane(15 + 8, 1); pools[10] = plane(15 + 12, 1);
}

// ---------------------------------------------------------------- prologue: Q-side rotation fold
// q'_g = Pi^(m_g) q_g * (scale*log2e/sqrt(m_g))  ("Q-side rotation"), rounded to fp16 and
// written in B-fragment order: qf[pair][kstep][head slot n (8)][c (4)][coords 2c, 2c+1, 8+2c, 9+2c], i.e. one
// 8-byte load per lane (n*4+c) and k-step; zero padded.
// Latency-shaped (it sits on the critical path of every decode call, 8.6 us per layer before): four threads share one
// output -- thread part p takes k = p, p+4, ... -- so that a group of up to 64 coordinates needs ONE round of 16 independent
// rotation loads per thread instead of four, and the ragged tail is a masked round instead of a serial loop.
// PARTS = 1 (one thread per output) serves the launches with many blocks, where throughput counts.
template <int PARTS>
__global__ void __launch_bounds__(PARTS * kDh)
qfold_kernel(const HeadMeta *__restrict__ metas, const float *__restrict__ rot_t,
             const __nv_bfloat16 *__restrict__ q, int batch, int Hkv, int Hq, float scale_log2e,
             __half *__restrict__ qf, int plain, int early_wait = 0)
{
    pdl_trigger();
    const int G = Hq / Hkv;
    const int pair = blockIdx.x / G, n = blockIdx.x % G;   // one block per (pair, query head of the group)
    const int h = pair % Hkv, lb = pair / Hkv, l = lb / batch;
    __shared__ __align__(8) HeadMeta Ms;                    // one coalesced copy: the k-step scan and the group search below
    __shared__ float qs[kDh];                               // were chains of dependent global loads on the critical path
    __shared__ int ksbase[kMaxGroups];
    const int tid = threadIdx.x;
    {
        const uint32_t *msrc = reinterpret_cast<const uint32_t *>(metas + l * Hkv + h);
        if (tid < (int)(sizeof(HeadMeta) / 4)) reinterpret_cast<uint32_t *>(&Ms)[tid] = __ldg(msrc + tid);
    }
    constexpr int kQfoldThreads = PARTS * kDh;
    constexpr int q0 = PARTS > 1 ? kDh : 0;                 // (another warp set than the metadata copy)
    if (tid >= q0 && tid < q0 + kDh) qs[tid - q0] = __bfloat162float(q[((size_t)lb * Hq + h * G + n) * kDh + tid - q0]);
    __syncthreads();
    const HeadMeta &M = Ms;
    if (tid == 0)
        for (int ks = 0; ks < M.n_ksteps; ++ks)
            if (M.ksteps[ks].flags & 1) ksbase[M.ksteps[ks].flags >> 4] = ks;
    __syncthreads();                                        // ksbase[]
    // plain layout (prefill): q'[pair][head slot n][128] in grouped coordinate order, zero beyond kdim
    if (plain && tid < kDh && tid >= M.kdim) qf[((size_t)pair * 8 + n) * kDh + tid] = __float2half(0.f);
    const int ro = tid / PARTS, part = tid % PARTS;         // output (grouped coordinate) and the part of its dot product
    const bool act = ro < M.kdim;
    float acc = 0.f, sc = 0.f;
    int ks = 0, kap = 0;
    if (act) {
        int g = 0;
        while (g + 1 < M.n_groups && ro >= M.gstart[g + 1]) ++g;
        const int m = M.gm[g], x0 = M.gstart[g], r = ro - x0;
        const float *T = rot_t + rot_offset(m) + r;
        sc = scale_log2e / sqrtf((float)m) * (BGTQ_NORM_IN_OPERAND ? 64.f : 1.f);   // 2^6: see qk_group_n
        ks = ksbase[g] + (r >> 4); kap = r & 15;
        const uint8_t *co = M.coords + x0;
        if constexpr (PARTS == 1) {                         // throughput form: full rounds unmasked, scalar tail
            int k = 0;
            for (; k + 16 <= m; k += 16) {
                float tv[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) tv[u] = __ldg(T + (size_t)(k + u) * m);
#pragma unroll
                for (int u = 0; u < 16; ++u) acc = fmaf(tv[u], qs[co[k + u]], acc);
            }
            for (; k < m; ++k) acc = fmaf(__ldg(T + (size_t)k * m), qs[co[k]], acc);
        } else {
            for (int k0 = 0; k0 < m; k0 += 16 * PARTS) {    // 16 independent rotation loads in flight per thread, masked tail round
                float tv[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) { const int k = k0 + part + PARTS * u; tv[u] = k < m ? __ldg(T + (size_t)k * m) : 0.f; }
#pragma unroll
                for (int u = 0; u < 16; ++u) { const int k = k0 + part + PARTS * u; acc = fmaf(tv[u], k < m ? qs[co[k]] : 0.f, acc); }
            }
        }
    }
#pragma unroll
    for (int sft = 1; sft < PARTS; sft <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, sft);   // the parts of an output are adjacent lanes; fixed order
    // Launched programmatically behind the previous decode call's combine_kernel (per-layer chains), this block has come
    // this far -- metadata, the query row (a caller input, complete before the call), the dot products -- beside it; the
    // q' workspace may still be read by that call's decode_kernel until its combine_kernel has completed.
    if (early_wait) pdl_wait();
    // zero padding: this head's slots (and, from block n = 0, the unused head slots n >= G)
    uint2 *out2 = reinterpret_cast<uint2 *>(qf + (size_t)pair * kQfHalves);     // [kstep][8][4] of 4 halves
    if (!plain)
        for (int e = tid; e < kMaxKSteps * 32; e += kQfoldThreads) {
            const int nn = (e >> 2) & 7;
            if (nn == n || (n == 0 && nn >= G)) out2[e] = make_uint2(0u, 0u);
        }
    __syncthreads();
    if (act && part == 0) {
        __half *out = qf + (size_t)pair * kQfHalves;
        if (plain) qf[((size_t)pair * 8 + n) * kDh + ro] = __float2half_rn(acc * sc);
        else out[((ks * 8 + n) * 4 + ((kap & 7) >> 1)) * 4 + (kap >> 3) * 2 + (kap & 1)] = __float2half_rn(acc * sc);
    }
    // Protected regime: this kernel is launched programmatically behind window_kernel and runs beside it; it must not
    // COMPLETE before window_kernel has, because the kernels after it only wait for their immediate predecessor.
    // (A no-op when the launch carries no programmatic dependency.)
    if (!early_wait) pdl_wait();
}

// ---------------------------------------------------------------- the decode kernel
struct DecodeParams {
    const HeadMeta *metas;      // [n_layers][Hkv], first layer of this call
    const uint8_t *cache;
    const __half *qf;           // q' fragments, [pair][kQfHalves]
    const int32_t *seq_len;
    const uint16_t *cb16;
    const uint16_t *hcb16;      // exact-density codebooks: [head of the call][2][kHeadLutHalves] (K, V), else nullptr
    float *partials;            // [n_warps + n_pairs][8][130]
    int64_t n_cap;              // tiles of capacity per sequence
    int n_layers, batch, Hkv, G;
    int buf_bytes;              // per-warp tile buffer
    const int32_t *pages;       // paged cache: [batch][pstride] page index per tile (nullptr: contiguous layout)
    int pstride;
    int64_t n_pages;
    int n_sink, n_recent;       // protected regime: packed tokens [n_sink, T - n_recent) only (0, 0 = the buffer-free path)
};

constexpr int kSmemHdr = 0;      // dynamic shared memory holds only the tile buffers (tables are static)
constexpr int kStaticSmem = 8 * 1024;   // upper bound of the kernel's static shared memory

// load the B words of one unit for this lane.  FULL: 32 lanes per word plane (stride 32 words).
template <int B>
__device__ __forceinline__ void load_unit_full(const uint32_t *unit, int lane, uint32_t (&w)[B])
{
#pragma unroll
    for (int i = 0; i < B; ++i) w[i] = unit[i * 32 + lane];
}
// trailing partial half-step: only lanes c < nc hold data, compacted to 8*nc lanes per plane
template <int B>
__device__ __forceinline__ void load_unit_partial(const uint32_t *unit, int g8, int c, int nc, uint32_t (&w)[B])
{
    const bool act = c < nc;
    const uint32_t *wp = unit + g8 * nc + c;
#pragma unroll
    for (int i = 0; i < B; ++i) w[i] = act ? wp[i * 8 * nc] : 0u;
}

// word i of this lane at unit[off + i * stride].  Full unit: off = lane, stride = 32.  The group's trailing partial unit
// (nc = 1..3 lanes per token row hold data, compacted to 8*nc lanes per plane): off = g8*nc + c, stride = 8*nc.  Lanes
// c >= nc read in-bounds words they do not own (the next plane, the next unit or the K norms that follow the codes in the
// same half-tile copy): whatever they decode is a finite codebook value and meets the zero rows of q' (qfold_kernel pads
// every k-step with zeros), so no predicate and no zero fill is needed.
template <int B>
__device__ __forceinline__ void load_unit_at(const uint32_t *unit, int off, int stride, uint32_t (&w)[B])
{
#pragma unroll
    for (int i = 0; i < B; ++i) w[i] = unit[off + i * stride];
}

// QK^T of one same-width group.  m = coordinates in the group; units of 8 coordinates are contiguous
// (128*B bytes each), only the last may be partial.  Units are taken in pairs (one m16n8k16 step per pair and m-tile); an
// odd last unit is one m16n8k8 step on the first half of its q' fragment.  The group's first step starts the
// accumulators (C = 0).
template <int B, bool P5>
__device__ __forceinline__ void qk_group(const uint32_t *gcodes, int m, int lane, const uint2 *__restrict__ qfp,
                                         const uint32_t *pools, const uint16_t *lut, float (&A)[8][4])
{
    const int g8 = lane >> 2, c = lane & 3;
    const int n_full = m >> 3, rem = (m & 7) >> 1, n_units = n_full + (rem ? 1 : 0);
    const int offp = rem ? g8 * rem + c : lane, strp = rem ? 8 * rem : 32;     // addressing of the group's LAST unit
    const uint32_t *u0 = gcodes;
    bool first = true;
#pragma unroll 1
    for (int p = n_units >> 1; p > 0; --p) {
        uint32_t w0[B], w1[B], h0[16], h1[16];
        const uint2 bq = __ldg(qfp);
        const bool last1 = p == 1 && !(n_units & 1);            // this pair's second unit is the group's last unit
        load_unit_full<B>(u0, lane, w0);
        load_unit_at<B>(u0 + 32 * B, last1 ? offp : lane, last1 ? strp : 32, w1);
        decode_unit<B, P5>(w0, pools, lut, h0);
        decode_unit<B, P5>(w1, pools, lut, h1);
        if (first) {
#pragma unroll
            for (int i = 0; i < 8; ++i) mma16816_z(A[i], h0[2 * i], h0[2 * i + 1], h1[2 * i], h1[2 * i + 1], bq.x, bq.y);
            first = false;
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) mma16816(A[i], h0[2 * i], h0[2 * i + 1], h1[2 * i], h1[2 * i + 1], bq.x, bq.y);
        }
        u0 += 64 * B;
        qfp += 32;
    }
    if (n_units & 1) {
        uint32_t w0[B], h0[16];
        const uint32_t b0 = __ldg(reinterpret_cast<const uint32_t *>(qfp));
        load_unit_at<B>(u0, offp, strp, w0);
        decode_unit<B, P5>(w0, pools, lut, h0);
        if (first) {
#pragma unroll
            for (int i = 0; i < 8; ++i) mma1688_z(A[i], h0[2 * i], h0[2 * i + 1], b0);
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) mma1688(A[i], h0[2 * i], h0[2 * i + 1], b0);
        }
    }
}

// Variant with the K group norm folded into the A operand (fp16): a *= n * 2^-6 before the MMA (q' carries the
// 2^6), so that ALL groups accumulate into one fp32 logit accumulator and no per-group fp32 scaling pass -- and
// no HMMA -> FFMA pipeline drain at every group boundary -- is needed.  nn[i][p] = (n, n) half2 of token row
// (16i + 8p + g8).  The product is rounded to fp16 (2^-11 relative), well inside the 2e-3 attention tolerance;
// the 2^-6 prescale keeps n * |c| <= 65504 * 4.6 / 64 finite for every fp16 norm.
__device__ __forceinline__ uint32_t hmul2_u(uint32_t a, uint32_t b)
{
    uint32_t r;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
template <int B, bool P5>
__device__ __forceinline__ void qk_group_n(const uint32_t *gcodes, int m, int lane, const uint2 *__restrict__ qfp,
                                           const uint32_t *pools, const uint16_t *lut, const uint32_t (&nn)[8][2],
                                           float (&S)[8][4])
{
    const int g8 = lane >> 2, c = lane & 3;
    const int n_full = m >> 3, rem = (m & 7) >> 1;
    const uint32_t *u0 = gcodes;
#pragma unroll 1
    for (int jp = n_full >> 1; jp > 0; --jp) {
        uint32_t w0[B], w1[B], h0[16], h1[16];
        const uint2 bq = __ldg(qfp);
        load_unit_full<B>(u0, lane, w0);
        load_unit_full<B>(u0 + 32 * B, lane, w1);
        decode_unit<B, P5>(w0, pools, lut, h0);
        decode_unit<B, P5>(w1, pools, lut, h1);
#pragma unroll
        for (int i = 0; i < 8; ++i)
            mma16816(S[i], hmul2_u(h0[2 * i], nn[i][0]), hmul2_u(h0[2 * i + 1], nn[i][1]),
                     hmul2_u(h1[2 * i], nn[i][0]), hmul2_u(h1[2 * i + 1], nn[i][1]), bq.x, bq.y);
        u0 += 64 * B;
        qfp += 32;
    }
    if ((n_full & 1) | rem) {
        uint32_t w0[B], h0[16], h1[16];
        const uint2 bq = __ldg(qfp);
        if (n_full & 1) load_unit_full<B>(u0, lane, w0);
        else load_unit_partial<B>(u0, g8, c, rem, w0);
        decode_unit<B, P5>(w0, pools, lut, h0);
        if ((n_full & 1) && rem) {
            uint32_t w1[B];
            load_unit_partial<B>(u0 + 32 * B, g8, c, rem, w1);
            decode_unit<B, P5>(w1, pools, lut, h1);
#pragma unroll
            for (int i = 0; i < 8; ++i)
                mma16816(S[i], hmul2_u(h0[2 * i], nn[i][0]), hmul2_u(h0[2 * i + 1], nn[i][1]),
                         hmul2_u(h1[2 * i], nn[i][0]), hmul2_u(h1[2 * i + 1], nn[i][1]), bq.x, bq.y);
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i)
                mma16816(S[i], hmul2_u(h0[2 * i], nn[i][0]), hmul2_u(h0[2 * i + 1], nn[i][1]), 0u, 0u, bq.x, bq.y);
        }
    }
}

// PV of one tile: 16 units of width B -> O[J] += V^T[16 dims x 128 tokens] . P[128 tokens x 8 heads]
// The eight k-steps of a block go to four accumulators (O[J] and three temporaries started with C = 0), so that four
// independent HMMAs are in flight instead of one chain of eight; the words of the next block are requested before the
// MMAs of the current one.
template <int B, bool P5>
__device__ __forceinline__ void pv_tile(const uint32_t *vcodes, int lane, const uint32_t (&bP)[8][2],
                                        const uint32_t *pools, const uint16_t *lut, float (&O)[8][4])
{
    uint32_t w0[B], w1[B];
    load_unit_full<B>(vcodes, lane, w0);
    load_unit_full<B>(vcodes + 32 * B, lane, w1);
#pragma unroll 1
    for (int J = 0; J < 8; ++J) {
        uint32_t h0[16], h1[16];
        decode_unit<B, P5>(w0, pools, lut, h0);
        decode_unit<B, P5>(w1, pools, lut, h1);
        if (J < 7) {
            const uint32_t *u0 = vcodes + (2 * J + 2) * 32 * B;
            load_unit_full<B>(u0, lane, w0);
            load_unit_full<B>(u0 + 32 * B, lane, w1);
        }
        float T[3][4];
        mma16816(O[J], h0[0], h1[0], h0[1], h1[1], bP[0][0], bP[0][1]);
#pragma unroll
        for (int kp = 1; kp < 4; ++kp)
            mma16816_z(T[kp - 1], h0[2 * kp], h1[2 * kp], h0[2 * kp + 1], h1[2 * kp + 1], bP[kp][0], bP[kp][1]);
        mma16816(O[J], h0[8], h1[8], h0[9], h1[9], bP[4][0], bP[4][1]);
#pragma unroll
        for (int kp = 5; kp < 8; ++kp)
            mma16816(T[kp - 5], h0[2 * kp], h1[2 * kp], h0[2 * kp + 1], h1[2 * kp + 1], bP[kp][0], bP[kp][1]);
#pragma unroll
        for (int e = 0; e < 4; ++e) O[J][e] += (T[0][e] + T[1][e]) + T[2][e];
    }
}

// PV of one 16-dimension V block (two units of width B): O0 += V^T[16 dims x 128 tokens] . P[128 tokens x 8 heads]
template <int B, bool P5>
__device__ __forceinline__ void pv_block(const uint32_t *u0, int lane, const uint32_t (&bP)[8][2],
                                         const uint32_t *pools, const uint16_t *lut, float (&O0)[4])
{
    uint32_t w0[B], w1[B], h0[16], h1[16];
    load_unit_full<B>(u0, lane, w0);
    load_unit_full<B>(u0 + 32 * B, lane, w1);
    decode_unit<B, P5>(w0, pools, lut, h0);
    decode_unit<B, P5>(w1, pools, lut, h1);
#pragma unroll
    for (int kp = 0; kp < 8; ++kp)
        mma16816(O0, h0[2 * kp], h1[2 * kp], h0[2 * kp + 1], h1[2 * kp + 1], bP[kp][0], bP[kp][1]);
}

// VG: heads may hold several V groups (V-side allocator, reading Q19): the accumulator and the partial record are in
// GROUPED V order (block J' of the record = original block vblk[J']), every V group brings its own norm row and width.
template <int W, bool PAGED, bool EXACT, bool VG>
__global__ void __launch_bounds__(W * 32, 1)
decode_kernel(const DecodeParams P)
{
    extern __shared__ __align__(128) unsigned char smem[];       // the per-warp tile buffers only
    constexpr bool P5 = !BGTQ_NO_P5;
    __shared__ __align__(16) uint16_t lut[P5 ? kLutHalves : 512]; // static: constant LDS addresses for the LUTs
    __shared__ uint32_t pools_s[W][2][12];                        // PRMT byte planes per warp: [0] K tables, [1] V table
    __shared__ int pre[kMaxBatch + 1];
    __shared__ __align__(8) uint64_t bars[2 * W];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g8 = lane >> 2, c = lane & 3;
    pdl_trigger();
#if BGTQ_TIMING
    unsigned long long tst[10];
    auto TS = [&](int i) { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tst[i])); };
    for (int i = 0; i < 10; ++i) tst[i] = 0;
    TS(0);
#else
    auto TS = [&](int) {};
#endif
    build_lut(P.cb16, lut, tid, W * 32, P5);
    if (tid == 0) build_prefix(P.seq_len, P.batch, P.n_cap * kTile, pre, P.n_sink, P.n_recent);
    __syncthreads();
    if (lane < 2 && !EXACT) build_pools(lut, pools_s[warp][lane]);   // shared codebooks: the same planes for every head
    const uint32_t *pools = pools_s[warp][0], *poolsV = pools_s[warp][1];
    const uint32_t kbar = smem_u32(&bars[2 * warp]), vbar = smem_u32(&bars[2 * warp + 1]);
    if (lane == 0) {
        mbar_init(kbar, 1);
        mbar_init(vbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    __syncthreads();
    TS(1);

    const int gw = blockIdx.x * W + warp;
    const Sched S = make_sched(P.n_layers, P.batch, P.Hkv, pre, gridDim.x, W);
    int x = warp_lo(S, blockIdx.x, warp);
    const int x_end = warp_lo(S, blockIdx.x, warp + 1);
    // CTA-level merge: when the whole CTA range lies inside one (layer, sequence, kv head) pair, the warps'
    // partials are merged in shared memory and ONE partial per CTA goes to HBM (slot of the CTA's warp 0).
    bool merged = false;
    int merged_pair = 0;
    {
        const int c_lo = cta_lo(S, blockIdx.x), c_hi = cta_lo(S, blockIdx.x + 1);
        if (c_lo < c_hi) {
            const TilePos tc = locate(c_lo, S, pre);
            merged = c_hi <= tc.pair_start + tc.tiles_b;
            merged_pair = tc.pair;
        }
    }
    if (!merged && x >= x_end) return;

    const uint32_t *tile = reinterpret_cast<const uint32_t *>(smem + kSmemHdr + warp * P.buf_bytes);
    const uint32_t tile_s = smem_u32(tile);
    uint32_t kphase = 0, vphase = 0;

    // lane 0 requests (a half of) a tile: K half = [K codes | K norms], V half = [V norms | V codes]
    // (the buffer was only READ through the generic proxy since its last fill, and __syncwarp orders those reads
    // before the copy is issued, so no cross-proxy fence is needed -- the usual consumer-release -> TMA pattern)
    auto issue_at = [&](const uint8_t *src, uint32_t kbytes, uint32_t vbytes, bool want_k, bool want_v) {
        if (want_k && kbytes) { mbar_expect_tx(kbar, kbytes); bulk_g2s(tile_s, src, kbytes, kbar); }   // (no K group: nothing to copy)
        if (want_v) { mbar_expect_tx(vbar, vbytes); bulk_g2s(tile_s + kbytes, src + kbytes, vbytes, vbar); }
    };
    auto tile_src = [&](const TilePos &tp, const HeadMeta &M) -> const uint8_t * {
        if (PAGED)
            return P.cache + P.n_pages * ((int64_t)M.layer_prefix + M.head_prefix) +
                   (int64_t)__ldg(P.pages + (int64_t)tp.b * P.pstride + tp.t) * M.tile_stride;
        return P.cache + P.n_cap * ((int64_t)P.batch * M.layer_prefix + (int64_t)tp.b * M.layer_sum + M.head_prefix) +
               (int64_t)tp.t * M.tile_stride;
    };
    if (x < x_end) {
        const TilePos tp0 = locate(x, S, pre);
        const HeadMeta &M0 = P.metas[tp0.l * P.Hkv + tp0.h];
        if (lane == 0) issue_at(tile_src(tp0, M0), M0.vnorm_off, M0.tile_stride - M0.vnorm_off, true, true);
    } else if (merged) {                       // idle warp of a merged CTA: contributes an empty partial
        float *rec = reinterpret_cast<float *>(smem + kSmemHdr + warp * P.buf_bytes);
        for (int i = lane; i < kPartialFloats; i += 32) rec[i] = (i % 130 == 0) ? -INFINITY : 0.f;
    }
    // The first tile is already in flight (the cache was complete before qfold_kernel started: it is launched without
    // the attribute); q' and the partial-record workspace may be touched only after the predecessor has completed.
    TS(2);
    pdl_wait();
    TS(3);

    while (x < x_end) {
        // ---------------- segment = the part of one (layer, sequence, kv head) inside this warp's range
        const TilePos tp = locate(x, S, pre);
        const HeadMeta &M = P.metas[tp.l * P.Hkv + tp.h];
        const int seg_end = min(x_end, tp.pair_start + tp.tiles_b);
        const int n_groups = M.n_groups, b_v = M.b_v;
        const int knorm_off = M.knorm_off, vnorm_off = M.vnorm_off, vcode_off = M.vcode_off;
        // codebook tables of this head: shared Gaussian tables in shared memory, or the head's exact-density tables
        // (global memory, L1-resident: 10 KB per head) with the byte planes rebuilt per segment
        const uint16_t *lutK = lut, *lutV = lut;
        if (EXACT) {
            lutK = P.hcb16 + (size_t)(tp.l * P.Hkv + tp.h) * 2 * kHeadLutHalves;
            lutV = lutK + kHeadLutHalves;
            __syncwarp();
            if (lane < 2) build_pools(lane ? lutV : lutK, pools_s[warp][lane]);
            __syncwarp();
        }
        int64_t slen = P.seq_len[tp.b];
        slen = slen > P.n_cap * kTile ? P.n_cap * kTile : slen;
        slen = packed_len(slen, P.n_sink, P.n_recent);
        // lane g keeps the descriptor of group g: code offset | m << 16 | b << 24 | first k-step << 28
        uint32_t gdesc = 0;
        if (lane < n_groups) {
            int ksb = 0;
            for (int g = 0; g < lane; ++g) ksb += (M.gm[g] + 15) >> 4;
            gdesc = (uint32_t)M.goff[lane] | ((uint32_t)(M.gm[lane] & 0xFF) << 16) | ((uint32_t)M.gb[lane] << 24) | ((uint32_t)ksb << 28);
        }
        // lane J' keeps the descriptor of grouped V block J': unit offset | width << 16 | V group << 20 | first of its group << 24
        uint32_t vdesc = 0;
        if (VG && lane < kMaxGroups) {
            const int gv = M.vbg[lane];
            vdesc = (uint32_t)M.vboff[lane] | ((uint32_t)M.vbw[lane] << 16) | ((uint32_t)gv << 20) | (M.vgstart[gv] == lane ? 1u << 24 : 0u);
        }
        const uint2 *qfp = reinterpret_cast<const uint2 *>(P.qf + (size_t)tp.pair * kQfHalves) + lane;
        const uint8_t *src = tile_src(tp, M);                     // current tile of this segment (advanced per tile)
        const uint32_t stride = M.tile_stride, kbytes = M.vnorm_off, vbytes = stride - kbytes;
        const uint8_t *pool = P.cache + P.n_pages * ((int64_t)M.layer_prefix + M.head_prefix);   // paged layout only
        const int32_t *prow = P.pages + (int64_t)tp.b * P.pstride;

        float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;   // heads 2c, 2c+1 (log2 domain)
        float O[8][4];
#pragma unroll
        for (int J = 0; J < 8; ++J) O[J][0] = O[J][1] = O[J][2] = O[J][3] = 0.f;

        for (int t = tp.t; x < seg_end; ++x, ++t) {
            // ======== QK^T
            // paged: the next tile's page index is fetched a whole QK^T ahead of the copy that needs it
            const int next_page = (PAGED && x + 1 < seg_end) ? __ldg(prow + t + 1) : 0;
            if (kbytes) { mbar_wait(kbar, kphase); kphase ^= 1; }
            TS(4);
            float Sc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i) Sc[i][0] = Sc[i][1] = Sc[i][2] = Sc[i][3] = 0.f;
#pragma unroll 1
            for (int g = 0; g < n_groups; ++g) {
                const uint32_t d = __shfl_sync(0xFFFFFFFFu, gdesc, g);
                int m = (d >> 16) & 0xFF;
                m = m ? m : 128;
                const uint32_t *gcodes = tile + ((d & 0xFFFF) >> 2);
                const uint2 *qg = qfp + (d >> 28) * 32;
#if BGTQ_NORM_IN_OPERAND
                // group norms (fp16, pre-scaled by 2^-6) duplicated to (n, n) pairs and folded into the A operand
                const uint4 *np = reinterpret_cast<const uint4 *>(tile + ((knorm_off + 256 * g + g8 * 32) >> 2));
                const uint4 n0 = np[0], n1 = np[1];
                const uint32_t nw[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
                uint32_t nn[8][2];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const uint32_t xs = hmul2_u(nw[i], 0x24002400u);       // * 2^-6 (exact)
                    nn[i][0] = prmt(xs, xs, 0x1010);
                    nn[i][1] = prmt(xs, xs, 0x3232);
                }
                switch ((d >> 24) & 0xF) {
                case 1: qk_group_n<1, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                case 2: qk_group_n<2, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                case 3: qk_group_n<3, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                case 4: qk_group_n<4, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                case 5: qk_group_n<5, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                case 6: qk_group_n<6, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                case 7: qk_group_n<7, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                default: qk_group_n<8, P5>(gcodes, m, lane, qg, pools, lutK, nn, Sc); break;
                }
            }
#else
                float A[8][4];                               // started by the group's first k-step (m >= 2)
                switch ((d >> 24) & 0xF) {
                case 1: qk_group<1, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                case 2: qk_group<2, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                case 3: qk_group<3, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                case 4: qk_group<4, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                case 5: qk_group<5, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                case 6: qk_group<6, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                case 7: qk_group<7, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                default: qk_group<8, P5>(gcodes, m, lane, qg, pools, lutK, A); break;
                }
                // scale by the fp16 group norms (fp32, on the accumulators)
                const uint4 *np = reinterpret_cast<const uint4 *>(tile + ((knorm_off + 256 * g + g8 * 32) >> 2));
                const uint4 n0 = np[0], n1 = np[1];
                const uint32_t nw[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float2 nf = __half22float2(*reinterpret_cast<const __half2 *>(&nw[i]));
                    Sc[i][0] = fmaf(nf.x, A[i][0], Sc[i][0]);
                    Sc[i][1] = fmaf(nf.x, A[i][1], Sc[i][1]);
                    Sc[i][2] = fmaf(nf.y, A[i][2], Sc[i][2]);
                    Sc[i][3] = fmaf(nf.y, A[i][3], Sc[i][3]);
                }
            }
#endif
            __syncwarp();
            src = PAGED ? pool + (int64_t)next_page * stride : src + stride;
            if (lane == 0 && x + 1 < seg_end) issue_at(src, kbytes, vbytes, true, false);   // K half of the next tile (same layout only)

            TS(5);
            // ======== mask the ragged tail, online softmax (log2 domain)
            const int n_valid = (int)min((int64_t)kTile, slen - (int64_t)t * kTile);
            const int n_low = t == 0 ? P.n_sink : 0;           // sink tokens are served by the fp16 window (tile 0 only)
            if (n_valid < kTile || n_low > 0) {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int r0 = 16 * i + g8, r1 = r0 + 8;
                    if (r0 >= n_valid || r0 < n_low) Sc[i][0] = Sc[i][1] = -INFINITY;
                    if (r1 >= n_valid || r1 < n_low) Sc[i][2] = Sc[i][3] = -INFINITY;
                }
            }
            float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                mx0 = fmaxf(mx0, fmaxf(Sc[i][0], Sc[i][2]));
                mx1 = fmaxf(mx1, fmaxf(Sc[i][1], Sc[i][3]));
            }
#pragma unroll
            for (int o = 4; o < 32; o <<= 1) {
                mx0 = fmaxf(mx0, __shfl_xor_sync(0xFFFFFFFFu, mx0, o));
                mx1 = fmaxf(mx1, __shfl_xor_sync(0xFFFFFFFFu, mx1, o));
            }
            const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
            const float al0 = fast_exp2(m0 - mn0), al1 = fast_exp2(m1 - mn1);
            m0 = mn0; m1 = mn1;
            float ls0 = 0.f, ls1 = 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                Sc[i][0] = fast_exp2(Sc[i][0] - mn0); Sc[i][2] = fast_exp2(Sc[i][2] - mn0);
                Sc[i][1] = fast_exp2(Sc[i][1] - mn1); Sc[i][3] = fast_exp2(Sc[i][3] - mn1);
                ls0 += Sc[i][0] + Sc[i][2];
                ls1 += Sc[i][1] + Sc[i][3];
            }
            l0 = fmaf(l0, al0, ls0);
            l1 = fmaf(l1, al1, ls1);
            if (__any_sync(0xFFFFFFFFu, al0 != 1.f || al1 != 1.f)) {
#pragma unroll
                for (int J = 0; J < 8; ++J) { O[J][0] *= al0; O[J][2] *= al0; O[J][1] *= al1; O[J][3] *= al1; }
            }

            // ======== P * (V norm) -> fp16 B fragments (8x8 transposes), then PV
            mbar_wait(vbar, vphase);
            vphase ^= 1;
            TS(6);
            uint32_t bP[8][2];
            if constexpr (VG) {
#pragma unroll 1
                for (int Jg = 0; Jg < kMaxGroups; ++Jg) {
                    const uint32_t d = __shfl_sync(0xFFFFFFFFu, vdesc, Jg);
                    if (d >> 24) {                         // first block of a V group: P * (its norms) -> B fragments
                        const uint4 *np = reinterpret_cast<const uint4 *>(tile + ((vnorm_off + 256 * ((d >> 20) & 0xF) + g8 * 32) >> 2));
                        const uint4 n0 = np[0], n1 = np[1];
                        const uint32_t nw[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            const float2 nf = __half22float2(*reinterpret_cast<const __half2 *>(&nw[i]));
                            bP[i][0] = movmatrix_trans(pack_half2(Sc[i][0] * nf.x, Sc[i][1] * nf.x));
                            bP[i][1] = movmatrix_trans(pack_half2(Sc[i][2] * nf.y, Sc[i][3] * nf.y));
                        }
                    }
                    const uint32_t *u0 = tile + ((d & 0xFFFF) >> 2);
                    switch ((d >> 16) & 0xF) {
                    case 1: pv_block<1, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    case 2: pv_block<2, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    case 3: pv_block<3, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    case 4: pv_block<4, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    case 5: pv_block<5, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    case 6: pv_block<6, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    case 7: pv_block<7, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    default: pv_block<8, P5>(u0, lane, bP, poolsV, lutV, O[0]); break;
                    }
                    // rotate the accumulator blocks: after the eight blocks O is back in grouped order
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float t0 = O[0][e];
#pragma unroll
                        for (int J = 0; J < 7; ++J) O[J][e] = O[J + 1][e];
                        O[7][e] = t0;
                    }
                }
            } else {
                const uint4 *np = reinterpret_cast<const uint4 *>(tile + ((vnorm_off + g8 * 32) >> 2));
                const uint4 n0 = np[0], n1 = np[1];
                const uint32_t nw[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float2 nf = __half22float2(*reinterpret_cast<const __half2 *>(&nw[i]));
                    bP[i][0] = movmatrix_trans(pack_half2(Sc[i][0] * nf.x, Sc[i][1] * nf.x));
                    bP[i][1] = movmatrix_trans(pack_half2(Sc[i][2] * nf.y, Sc[i][3] * nf.y));
                }
            }
            if constexpr (!VG) {
                const uint32_t *vcodes = tile + (vcode_off >> 2);
                switch (b_v) {
                case 1: pv_tile<1, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                case 2: pv_tile<2, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                case 3: pv_tile<3, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                case 4: pv_tile<4, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                case 5: pv_tile<5, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                case 6: pv_tile<6, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                case 7: pv_tile<7, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                default: pv_tile<8, P5>(vcodes, lane, bP, poolsV, lutV, O); break;
                }
            }
            __syncwarp();
            TS(7);
            if (x + 1 < seg_end) {
                if (lane == 0) issue_at(src, kbytes, vbytes, false, true);                   // V half of the next tile
            } else if (x + 1 < x_end) {                                                      // next segment: other layout
                const TilePos tn = locate(x + 1, S, pre);
                const HeadMeta &Mn = P.metas[tn.l * P.Hkv + tn.h];
                if (lane == 0) issue_at(tile_src(tn, Mn), Mn.vnorm_off, Mn.tile_stride - Mn.vnorm_off, true, true);
            }
        }

        // ---------------- write this warp's partial for the pair: slot = warp + pair (unique, see combine)
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            l0 += __shfl_xor_sync(0xFFFFFFFFu, l0, o);
            l1 += __shfl_xor_sync(0xFFFFFFFFu, l1, o);
        }
        float *rec = merged ? reinterpret_cast<float *>(smem + kSmemHdr + warp * P.buf_bytes)
                            : P.partials + (size_t)(gw + tp.pair) * kPartialFloats;
        const int n0 = 2 * c, n1 = 2 * c + 1;
        if (n0 < P.G) {
            float *r0 = rec + n0 * 130;
            if (g8 == 0) { r0[0] = m0; r0[1] = l0; }
#pragma unroll
            for (int J = 0; J < 8; ++J) { r0[2 + 16 * J + g8] = O[J][0]; r0[2 + 16 * J + 8 + g8] = O[J][2]; }
        }
        if (n1 < P.G) {
            float *r1 = rec + n1 * 130;
            if (g8 == 0) { r1[0] = m1; r1[1] = l1; }
#pragma unroll
            for (int J = 0; J < 8; ++J) { r1[2 + 16 * J + g8] = O[J][1]; r1[2 + 16 * J + 8 + g8] = O[J][3]; }
        }
    }
    TS(8);
    if (merged) {      // exact log-sum-exp merge of the W warp partials, one record per CTA
        __syncthreads();
        const float *all = reinterpret_cast<const float *>(smem + kSmemHdr);
        const int fstride = P.buf_bytes >> 2;
        float *dst = P.partials + (size_t)(blockIdx.x * W + merged_pair) * kPartialFloats;
        for (int e = tid; e < 8 * 128; e += W * 32) {
            const int n = e >> 7, dd = e & 127;
            if (n >= P.G) continue;
            float Mx = -INFINITY;
#pragma unroll
            for (int w = 0; w < W; ++w) Mx = fmaxf(Mx, all[w * fstride + n * 130]);
            float acc = 0.f, ls = 0.f;
#pragma unroll
            for (int w = 0; w < W; ++w) {
                const float *r = all + w * fstride + n * 130;
                const float f = fast_exp2(r[0] - Mx);
                acc = fmaf(r[2 + dd], f, acc);
                ls = fmaf(r[1], f, ls);
            }
            dst[n * 130 + 2 + dd] = acc;
            if (dd == 0) { dst[n * 130] = Mx; dst[n * 130 + 1] = ls; }
        }
    }
#if BGTQ_TIMING
    TS(9);
    if (lane == 0 && (blockIdx.x % 37) == 5 && warp < 2)
        printf("cta %d warp %d: prologue %llu issue %llu pdlwait %llu ktile %llu qk %llu softmax+vwait %llu pv %llu tail %llu merge %llu total %llu\n", blockIdx.x, warp,
               tst[1] - tst[0], tst[2] - tst[1], tst[3] - tst[2], tst[4] - tst[3], tst[5] - tst[4], tst[6] - tst[5], tst[7] - tst[6], tst[8] - tst[7], tst[9] - tst[8], tst[9] - tst[0]);
#endif
}

// ---------------------------------------------------------------- a6: exact LSE merge + V de-rotation
// M = max_w m_w; l = sum_w l_w 2^(m_w-M); o' = sum_w acc_w 2^(m_w-M) / l, then
// out = Pi^(128)^T o' / sqrt(128)  (dequantisation of V, applied once because it is linear) -> bf16.
// Latency-shaped like qfold_kernel (it ends every decode call): 512 threads per (pair, query head), one record per thread in
// pass 1 (its running max and sum in one round trip), 16 warps over the records in pass 2, four threads per output
// dimension in the de-rotation.  Every reduction has a fixed order, so the result does not depend on timing.
// PARTS = 1 (128 threads) serves the launches with many blocks.
template <int PARTS>
__global__ void __launch_bounds__(PARTS * kDh)
combine_kernel(const float *__restrict__ partials, const int32_t *__restrict__ seq_len,
               const float *__restrict__ rot128, int n_layers, int batch, int Hkv, int G, int64_t n_cap,
               int n_ctas, int W, __nv_bfloat16 *__restrict__ out, int n_sink, int n_recent, int win_slot,
               const HeadMeta *__restrict__ metas, const float *__restrict__ rot_base)
{
    constexpr int kCombineThreads = PARTS * kDh;
    constexpr int kMaxSlots = 1024;                     // 32 + n_ctas entries at most (host checks n_ctas)
    constexpr int NW = kCombineThreads / 32;
    __shared__ int pre[kMaxBatch + 1];
    __shared__ float o[kDh];
    __shared__ int slots[kMaxSlots];
    __shared__ float wgt[kMaxSlots], lrec[kMaxSlots];
    __shared__ float red[NW][kDh + 4];
    __shared__ float wred[2][NW];
    pdl_trigger();                                      // the next decode call's qfold_kernel may run its prologue beside this kernel
    const int pair = blockIdx.x / G, n = blockIdx.x % G;
    const int h = pair % Hkv, lb = pair / Hkv, b = lb % batch, l = lb / batch;
    const int t = threadIdx.x, lane = t & 31, wq = t >> 5;
    const int d = t & (kDh - 1), part = t >> 7;         // de-rotation: output dimension and the part of its dot product
    if (t == 0) build_prefix(seq_len, batch, n_cap * kTile, pre, n_sink, n_recent);
    __syncthreads();
    const Sched S = make_sched(n_layers, batch, Hkv, pre, n_ctas, W);
    const int tiles_b = pre[b + 1] - pre[b];
    __nv_bfloat16 *dst = out + ((size_t)lb * Hkv * G + h * G + n) * kDh;
    // protected regime: one more record per pair, written by window_kernel at slot win_slot (relative to the pair's
    // base, like every slot below); it exists whenever the sequence is not empty
    const bool has_win = win_slot >= 0 && seq_len[b] > 0;
    if (tiles_b == 0 && !has_win) { if (t < kDh) dst[t] = __float2bfloat16(0.f); return; }
    const int start = l * (Hkv * S.tiles_sum) + pre[b] * Hkv + h * tiles_b, stop = start + tiles_b;
    // CTAs whose range meets [start, stop): the decode kernel's balanced split, recomputed
    int c0 = 0, c1 = 0;
    if (tiles_b > 0) {
        c0 = (int)(((int64_t)start * S.n_ctas) / S.total); c1 = (int)(((int64_t)(stop - 1) * S.n_ctas) / S.total);
        while (c0 + 1 < S.n_ctas && cta_lo(S, c0 + 1) <= start) ++c0;
        while (c0 > 0 && cta_lo(S, c0) > start) --c0;
        while (c1 + 1 < S.n_ctas && cta_lo(S, c1 + 1) <= stop - 1) ++c1;
        while (c1 > 0 && cta_lo(S, c1) > stop - 1) --c1;
    }
    // slot list in a fixed order: [warps of the first CTA][interior CTAs][warps of the last CTA].  Interior
    // CTAs lie wholly inside the pair, so they merged their warps (one record at the slot of warp 0); a CTA
    // straddling the pair boundary left one record per warp.
    const float *rec0 = partials + (size_t)pair * kPartialFloats + n * 130;
    auto edge_slot = [&](int c, int w) -> int {         // record of warp w of boundary CTA c, or -1
        const int lo = cta_lo(S, c), hi = cta_lo(S, c + 1);
        if (lo >= start && hi <= stop) return (w == 0 && lo < hi) ? c * W : -1;
        if (w >= W) return -1;
        const int wl = warp_lo(S, c, w), wh = warp_lo(S, c, w + 1);
        return (wl < wh && wl < stop && wh > start) ? c * W + w : -1;
    };
    const int n_int = c1 - c0 - 1 > 0 ? c1 - c0 - 1 : 0;
    const int n_pk = tiles_b > 0 ? min(kMaxSlots - 1, 16 + n_int + (c1 > c0 ? 16 : 0)) : 0;   // records of the packed range
    const int n_ent = n_pk + (has_win ? 1 : 0);
    // de-rotation operands of this thread (a static table): requested ahead of the wait, consumed after the merge
    constexpr int kRotPre = PARTS == 4 ? kDh / PARTS : 1;
    float rpre[kRotPre];
    if (PARTS == 4 && rot128 != nullptr && metas == nullptr) {
#pragma unroll
        for (int j = 0; j < kRotPre; ++j) rpre[j] = __ldg(rot128 + (part * kRotPre + j) * kDh + d);
    }
    pdl_wait();                                         // the decode kernel's partials are complete from here on
    // pass 1: every record's running max and sum (one round trip: the two loads are independent) -> M
    float mloc = -INFINITY;
    for (int e = t; e < n_ent; e += kCombineThreads) {
        const int sl = e >= n_pk ? win_slot
                     : e < 16 ? edge_slot(c0, e) : (e < 16 + n_int ? edge_slot(c0 + 1 + e - 16, 0) : edge_slot(c1, e - 16 - n_int));
        slots[e] = sl;
        const float2 ml = sl < 0 ? make_float2(-INFINITY, 0.f) : *reinterpret_cast<const float2 *>(rec0 + (size_t)sl * kPartialFloats);
        wgt[e] = ml.x;
        lrec[e] = ml.y;
        mloc = fmaxf(mloc, ml.x);
    }
#pragma unroll
    for (int s = 16; s; s >>= 1) mloc = fmaxf(mloc, __shfl_xor_sync(0xffffffffu, mloc, s));
    if (lane == 0) wred[0][wq] = mloc;
    __syncthreads();
    float Mx = wred[0][0];
#pragma unroll
    for (int w = 1; w < NW; ++w) Mx = fmaxf(Mx, wred[0][w]);
    // weights 2^(m - M) and the merged sum l
    float lloc = 0.f;
    for (int e = t; e < n_ent; e += kCombineThreads) {
        const float mw = wgt[e];
        const float f = (slots[e] < 0 || mw == -INFINITY) ? 0.f : exp2f(mw - Mx);
        wgt[e] = f;
        lloc = fmaf(lrec[e], f, lloc);
    }
#pragma unroll
    for (int s = 16; s; s >>= 1) lloc += __shfl_xor_sync(0xffffffffu, lloc, s);
    if (lane == 0) wred[1][wq] = lloc;
    __syncthreads();
    float lsum = 0.f;
#pragma unroll
    for (int w = 0; w < NW; ++w) lsum += wred[1][w];
    // pass 2: warp wq accumulates records wq, wq+16, ...; a lane owns dims 2*lane, 2*lane+1, 64+2*lane, 65+2*lane
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll 4
    for (int e = wq; e < n_ent; e += NW) {
        const float f = wgt[e];
        if (f == 0.f) continue;
        const float *rec = rec0 + (size_t)slots[e] * kPartialFloats + 2;
        const float2 lo = *reinterpret_cast<const float2 *>(rec + 2 * lane);
        const float2 hi = *reinterpret_cast<const float2 *>(rec + 64 + 2 * lane);
        a0 = fmaf(lo.x, f, a0); a1 = fmaf(lo.y, f, a1); a2 = fmaf(hi.x, f, a2); a3 = fmaf(hi.y, f, a3);
    }
    red[wq][2 * lane] = a0; red[wq][2 * lane + 1] = a1; red[wq][64 + 2 * lane] = a2; red[wq][65 + 2 * lane] = a3;
    __syncthreads();
    if (t < kDh) {
        float acc = 0.f;
#pragma unroll
        for (int w = 0; w < NW; ++w) acc += red[w][t];
        o[t] = acc / lsum;
    }
    __syncthreads();
    if (rot128 == nullptr && metas == nullptr) { if (t < kDh) dst[t] = __float2bfloat16(o[t]); return; }   // fp16-cache comparison path: no rotation
    // de-rotation of output dimension d: four threads take a quarter of the dot product each (32 independent loads)
    float r = 0.f, inv = 0.08838834764831845f;          // 1/sqrt(128)
    int od = d;
    if (metas) {
        // V-side groups (reading Q19): record position d is grouped V coordinate d.  Its group of m coordinates starts at
        // s: out[coord(d)] = sum_j Pi^(m)[j][d - s] o[s + j] / sqrt(m), coord(d) = 16 * vblk[d >> 4] + (d & 15).
        const HeadMeta &M = metas[l * Hkv + h];
        const int gv = M.vbg[d >> 4], s = 16 * M.vgstart[gv], m = 16 * M.vgcnt[gv], mq = m / PARTS;
        const float *R = rot_base + rot_offset(m) + (d - s);
#pragma unroll 4
        for (int j = part * mq; j < (part + 1) * mq; ++j) r = fmaf(__ldg(R + j * m), o[s + j], r);
        inv = rsqrtf((float)m);
        od = 16 * M.vblk[d >> 4] + (d & 15);
    } else {
        if (PARTS == 4) {
#pragma unroll
            for (int j = 0; j < kRotPre; ++j) r = fmaf(rpre[j], o[part * kRotPre + j], r);
        } else {
#pragma unroll 32
            for (int j = part * (kDh / PARTS); j < (part + 1) * (kDh / PARTS); ++j) r = fmaf(__ldg(rot128 + j * kDh + d), o[j], r);
        }
    }
    if (PARTS == 1) { dst[od] = __float2bfloat16(r * inv); return; }
    red[part][d] = r;
    __syncthreads();
    if (t < kDh) dst[od] = __float2bfloat16(((red[0][t] + red[1][t]) + (red[2][t] + red[3][t])) * inv);
}

// ---------------------------------------------------------------- protected regime: fp16 sink / recent windows
// PAPER.md:286, 813-815 "[sink (fp16) | compressed | recent (fp16)]".  win_k, win_v: fp16
// [layer][sequence][kv head][n_sink + n_recent][128]; slot j < n_sink holds token j, slot n_sink + (t mod n_recent)
// holds token t >= n_sink while it is among the last n_recent (a ring: attention does not depend on the order).
// One CTA per (pair, query head) attends over the valid slots and leaves ONE partial record in the decode kernel's
// format -- running max and sum in the log2 domain, accumulator in the rotated V domain scaled by sqrt(128), i.e.
// acc = sqrt(128) Pi (sum_t p_t v_t), so that combine_kernel's Pi^T acc / sqrt(128) returns sum_t p_t v_t -- which
// combine_kernel merges with the packed range's records by the same exact log-sum-exp rule.
constexpr int kMaxWindow = 1024;                    // n_sink + n_recent upper bound (shared-memory logits; >= 4 * 128 for the reuse below)
__device__ __forceinline__ bool window_slot_valid(int s, int64_t T, int n_sink, int n_recent)
{
    if (s < n_sink) return s < T;
    const int64_t x = T - 1 - (s - n_sink);         // T-1 - r; the newest token congruent to r is T-1 - (x mod n_recent)
    if (x < 0) return false;
    return T - 1 - (x % n_recent) >= n_sink;
}
__global__ void __launch_bounds__(128)
window_kernel(const __half *__restrict__ win_k, const __half *__restrict__ win_v, const __nv_bfloat16 *__restrict__ q,
              const int32_t *__restrict__ seq_len, const float *__restrict__ rot128_t, float *__restrict__ partials,
              int batch, int Hkv, int G, int64_t n_cap, int n_sink, int n_recent, float scale_log2e, int win_slot,
              const HeadMeta *__restrict__ metas = nullptr, const float *__restrict__ rot_t_base = nullptr)
{
    __shared__ float lg[kMaxWindow];
    __shared__ float qs[kDh], o[kDh];
    __shared__ float red[4];
    pdl_trigger();                                      // qfold_kernel may run beside this kernel (it reads nothing of ours)
    const int pair = blockIdx.x / G, n = blockIdx.x % G;
    const int h = pair % Hkv, lb = pair / Hkv, b = lb % batch;
    const int d = threadIdx.x, lane = d & 31, wq = d >> 5;
    const int n_win = n_sink + n_recent;
    int64_t T = seq_len[b];
    T = T < 0 ? 0 : (T > n_cap * kTile ? n_cap * kTile : T);
    qs[d] = __bfloat162float(q[((size_t)lb * Hkv * G + h * G + n) * kDh + d]) * scale_log2e;
    __syncthreads();
    const __half *kw = win_k + (size_t)pair * n_win * kDh, *vw = win_v + (size_t)pair * n_win * kDh;
    // logits: one thread per slot, the whole 256-byte key row in sixteen independent 16-byte loads (one memory latency per
    // slot instead of one per load); q is read from shared memory (broadcast)
    float mloc = -INFINITY;
    for (int s = d; s < n_win; s += 128) {
        float v = -INFINITY;
        if (window_slot_valid(s, T, n_sink, n_recent)) {
            const uint4 *row = reinterpret_cast<const uint4 *>(kw + (size_t)s * kDh);
            uint4 raw[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) raw[c] = __ldg(row + c);
            float a0 = 0.f, a1 = 0.f;
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const uint32_t wds[4] = {raw[c].x, raw[c].y, raw[c].z, raw[c].w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&wds[e]));
                    a0 = fmaf(f.x, qs[8 * c + 2 * e], a0);
                    a1 = fmaf(f.y, qs[8 * c + 2 * e + 1], a1);
                }
            }
            v = a0 + a1;
        }
        lg[s] = v;
        mloc = fmaxf(mloc, v);
    }
#pragma unroll
    for (int sft = 16; sft; sft >>= 1) mloc = fmaxf(mloc, __shfl_xor_sync(0xffffffffu, mloc, sft));
    if (lane == 0) red[wq] = mloc;
    __syncthreads();
    const float Mx = fmaxf(fmaxf(red[0], red[1]), fmaxf(red[2], red[3]));
    float *rec = partials + (size_t)(win_slot + pair) * kPartialFloats + n * 130;
    // (launched programmatically behind the previous call's combine_kernel, which may still read the record workspace:
    //  every write to it comes after a griddepcontrol.wait -- a no-op without a programmatic dependency)
    if (Mx == -INFINITY) {                              // empty sequence: an empty record
        pdl_wait();
        if (d == 0) { rec[0] = -INFINITY; rec[1] = 0.f; }
        rec[2 + d] = 0.f;
        return;
    }
    // weights 2^(logit - max) in place (0 for an empty slot).  Then warp wq takes slots wq, wq+4, ... and a lane four
    // dimensions (one 8-byte load per slot), 32 slots' loads in flight at a time -- the value loads do not depend on the
    // weights; an empty slot's row may hold anything and is replaced by 0.  The four warps' partial sums meet in shared
    // memory in a fixed order.
    for (int s = d; s < n_win; s += 128) lg[s] = lg[s] == -INFINITY ? 0.f : fast_exp2(lg[s] - Mx);
    __syncthreads();
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, lw = 0.f;
    for (int s0 = wq; s0 < n_win; s0 += 4 * 32) {
        uint2 raw[32];
#pragma unroll
        for (int u = 0; u < 32; ++u) {
            const int s = s0 + 4 * u;
            raw[u] = s < n_win ? __ldg(reinterpret_cast<const uint2 *>(vw + (size_t)s * kDh + 4 * lane)) : make_uint2(0u, 0u);
        }
#pragma unroll
        for (int u = 0; u < 32; ++u) {
            const int s = s0 + 4 * u;
            const float pw = s < n_win ? lg[s] : 0.f;
            const float2 x = __half22float2(*reinterpret_cast<const __half2 *>(&raw[u].x));
            const float2 y = __half22float2(*reinterpret_cast<const __half2 *>(&raw[u].y));
            const bool on = pw != 0.f;
            lw += pw;
            a0 = fmaf(pw, on ? x.x : 0.f, a0); a1 = fmaf(pw, on ? x.y : 0.f, a1);
            a2 = fmaf(pw, on ? y.x : 0.f, a2); a3 = fmaf(pw, on ? y.y : 0.f, a3);
        }
    }
    float *part = lg;                                   // the logits are dead from here on: reuse as [4][128] + [4]
    __syncthreads();
    part[wq * kDh + 4 * lane] = a0; part[wq * kDh + 4 * lane + 1] = a1;
    part[wq * kDh + 4 * lane + 2] = a2; part[wq * kDh + 4 * lane + 3] = a3;
    if (lane == 0) red[wq] = lw;
    __syncthreads();
    const float lsum = (red[0] + red[1]) + (red[2] + red[3]);
    o[d] = (part[d] + part[kDh + d]) + (part[2 * kDh + d] + part[3 * kDh + d]);
    __syncthreads();
    if (metas) {
        // V-side groups: the record is in grouped V order, each group rotated by its own Pi^(m) and scaled by sqrt(m):
        // rec[s + r] = sqrt(m) sum_u Pi^(m)[r][u] o[coord(s + u)]  (the inverse of combine_kernel's per-group de-rotation)
        const HeadMeta &M = metas[(lb / batch) * Hkv + h];
        const int gv = M.vbg[d >> 4], s = 16 * M.vgstart[gv], m = 16 * M.vgcnt[gv];
        const float *T = rot_t_base + rot_offset(m) + (d - s);
        float r = 0.f;
#pragma unroll 16
        for (int u = 0; u < m; ++u) r = fmaf(__ldg(T + u * m), o[16 * M.vblk[(s + u) >> 4] + (u & 15)], r);
        pdl_wait();
        rec[2 + d] = r * sqrtf((float)m);
        if (d == 0) { rec[0] = Mx; rec[1] = lsum; }
        return;
    }
    float r = 0.f;                                      // acc_rot[d] = sqrt(128) * sum_j Pi[d][j] o[j]; rot128_t[j][d] = Pi[d][j]
#pragma unroll 32
    for (int j = 0; j < kDh; ++j) r = fmaf(__ldg(rot128_t + j * kDh + d), o[j], r);
    pdl_wait();
    rec[2 + d] = r * 11.313708498984761f;
    if (d == 0) { rec[0] = Mx; rec[1] = lsum; }
}

// fp16 copies of new tokens into the window buffers (the protected regime's companion of quantize_append): token i of the
// call sits at position seq_len[b] + i; it is stored iff it is a sink token or one of the call's last n_recent tokens
// (earlier ones would be overwritten inside the same call).  k_new, v_new [n_layers][batch][n_new][Hkv][128], fp32 or bf16.
template <typename T>
__global__ void __launch_bounds__(128)
window_append_kernel(const T *__restrict__ k_new, const T *__restrict__ v_new, const int32_t *__restrict__ seq_len,
                     __half *__restrict__ win_k, __half *__restrict__ win_v, int batch, int n_new, int Hkv,
                     int n_sink, int n_recent, int64_t max_tokens)
{
    const int i = blockIdx.x % n_new, lb = blockIdx.x / n_new, b = lb % batch, d = threadIdx.x;
    const int64_t t0 = seq_len[b], t = t0 + i;
    if (t >= max_tokens) return;                              // dropped by the append as well (capacity)
    const int64_t n_kept = min((int64_t)n_new, max_tokens - t0);   // tokens of this call that are cached
    int slot;
    if (t < n_sink) slot = (int)t;
    else if (n_recent > 0 && i >= n_kept - n_recent) slot = n_sink + (int)(t % n_recent);
    else return;
    const int n_win = n_sink + n_recent;
    for (int h = 0; h < Hkv; ++h) {
        const size_t src = (((size_t)lb * n_new + i) * Hkv + h) * kDh + d;
        const size_t dst = (((size_t)lb * Hkv + h) * n_win + slot) * kDh + d;
        win_k[dst] = __float2half_rn((float)k_new[src]);
        win_v[dst] = __float2half_rn((float)v_new[src]);
    }
}

// ---------------------------------------------------------------- comparison path: fp16 KV cache
// Not part of the method: an own split-KV decode kernel over a plain fp16 cache
// k_cache, v_cache [layer][sequence][kv head][token][128], same scheduler, same partial/combine format,
// so that "packed Block-GTQ cache vs fp16 cache" can be restated on this box without any
// third-party system.  HBM-bound by construction: 512 bytes per token per KV head.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}

struct Fp16Params {
    const __half *k_cache, *v_cache;
    const __nv_bfloat16 *q;     // [n_layers][batch][Hq][128]
    const int32_t *seq_len;
    float *partials;
    int64_t n_cap;
    int n_layers, batch, Hkv, G;
    float scale_log2e;
};

constexpr int kSubTok = 32;                       // tokens per staged sub-tile (4 per 128-token scheduling tile)
constexpr int kFp16Warps = 12;
constexpr int kFp16Buf = 2 * kSubTok * kDh * 2;   // K and V sub-tile, 16 KB per warp

__global__ void __launch_bounds__(kFp16Warps * 32, 1)
fp16_decode_kernel(const Fp16Params P)
{
    constexpr int W = kFp16Warps;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ int pre[kMaxBatch + 1];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g8 = lane >> 2, c = lane & 3;
    if (tid == 0) build_prefix(P.seq_len, P.batch, P.n_cap * kTile, pre);
    __syncthreads();
    const Sched S = make_sched(P.n_layers, P.batch, P.Hkv, pre, gridDim.x, W);
    int x = warp_lo(S, blockIdx.x, warp);
    const int x_end = warp_lo(S, blockIdx.x, warp + 1);
    bool merged = false;
    int merged_pair = 0;
    {
        const int c_lo = cta_lo(S, blockIdx.x), c_hi = cta_lo(S, blockIdx.x + 1);
        if (c_lo < c_hi) {
            const TilePos tc = locate(c_lo, S, pre);
            merged = c_hi <= tc.pair_start + tc.tiles_b;
            merged_pair = tc.pair;
        }
    }
    if (!merged && x >= x_end) return;
    unsigned char *buf = smem + warp * kFp16Buf;
    const uint32_t kbuf = smem_u32(buf), vbuf = kbuf + kSubTok * kDh * 2;
    const int gw = blockIdx.x * W + warp;
    if (x >= x_end) {
        float *rec = reinterpret_cast<float *>(buf);
        for (int i = lane; i < kPartialFloats; i += 32) rec[i] = (i % 130 == 0) ? -INFINITY : 0.f;
    }
    // stage 32 tokens x 128 halves with a 16-byte-chunk XOR swizzle (chunk ^= token & 7): conflict-free ldmatrix
    auto stage = [&](uint32_t dst, const __half *src) {      // src: first token of the sub-tile, row pitch 256 B
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int ch = i * 32 + lane, tok = ch >> 4, cc = ch & 15;
            cp_async16(dst + tok * 256 + ((cc ^ (tok & 7)) << 4), src + tok * kDh + cc * 8);
        }
    };
    while (x < x_end) {
        const TilePos tp = locate(x, S, pre);
        const int seg_end = min(x_end, tp.pair_start + tp.tiles_b);
        int64_t slen = P.seq_len[tp.b];
        slen = slen > P.n_cap * kTile ? P.n_cap * kTile : slen;
        const size_t row0 = ((size_t)tp.pair * P.n_cap * kTile) * kDh;       // pair = (l*batch+b)*Hkv+h
        const __half *kp = P.k_cache + row0, *vp = P.v_cache + row0;
        // q fragments: B[k = dim][n = head]; lane (n = g8, c) holds dims 16ks+2c,+1 and 16ks+8+2c,+1
        uint32_t bq[8][2];
        {
            const int l = tp.pair / (P.batch * P.Hkv), b = (tp.pair / P.Hkv) % P.batch, h = tp.pair % P.Hkv;
            const __nv_bfloat16 *qh = P.q + (((size_t)l * P.batch + b) * P.Hkv * P.G + h * P.G + g8) * kDh;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    float a = 0.f, bb = 0.f;
                    if (g8 < P.G) {
                        a = __bfloat162float(qh[16 * ks + 8 * hf + 2 * c]) * P.scale_log2e;
                        bb = __bfloat162float(qh[16 * ks + 8 * hf + 2 * c + 1]) * P.scale_log2e;
                    }
                    bq[ks][hf] = pack_half2(a, bb);
                }
        }
        float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
        float O[8][4];
#pragma unroll
        for (int J = 0; J < 8; ++J) O[J][0] = O[J][1] = O[J][2] = O[J][3] = 0.f;
        const int64_t tok_lo = (int64_t)tp.t * kTile, tok_hi = min(slen, (int64_t)(tp.t + (seg_end - x)) * kTile);
        const int n_sub = (int)((tok_hi - tok_lo + kSubTok - 1) / kSubTok);
        stage(kbuf, kp + tok_lo * kDh);
        asm volatile("cp.async.commit_group;" ::: "memory");
        stage(vbuf, vp + tok_lo * kDh);
        asm volatile("cp.async.commit_group;" ::: "memory");
        for (int s = 0; s < n_sub; ++s) {
            const int64_t t0 = tok_lo + (int64_t)s * kSubTok;
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            __syncwarp();
            float Sc[2][4];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                Sc[i][0] = Sc[i][1] = Sc[i][2] = Sc[i][3] = 0.f;
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    uint32_t a[4];
                    const int tok = 16 * i + (lane & 7) + 8 * ((lane >> 3) & 1), ch = 2 * ks + (lane >> 4);
                    ldmatrix_x4(a, kbuf + tok * 256 + ((ch ^ (tok & 7)) << 4));
                    mma16816(Sc[i], a[0], a[1], a[2], a[3], bq[ks][0], bq[ks][1]);
                }
            }
            __syncwarp();
            if (s + 1 < n_sub) stage(kbuf, kp + (t0 + kSubTok) * kDh);
            asm volatile("cp.async.commit_group;" ::: "memory");
            const int n_valid = (int)min((int64_t)kSubTok, slen - t0);
            if (n_valid < kSubTok) {
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    if (16 * i + g8 >= n_valid) Sc[i][0] = Sc[i][1] = -INFINITY;
                    if (16 * i + 8 + g8 >= n_valid) Sc[i][2] = Sc[i][3] = -INFINITY;
                }
            }
            float mx0 = fmaxf(fmaxf(Sc[0][0], Sc[0][2]), fmaxf(Sc[1][0], Sc[1][2]));
            float mx1 = fmaxf(fmaxf(Sc[0][1], Sc[0][3]), fmaxf(Sc[1][1], Sc[1][3]));
#pragma unroll
            for (int o = 4; o < 32; o <<= 1) {
                mx0 = fmaxf(mx0, __shfl_xor_sync(0xFFFFFFFFu, mx0, o));
                mx1 = fmaxf(mx1, __shfl_xor_sync(0xFFFFFFFFu, mx1, o));
            }
            const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
            const float al0 = fast_exp2(m0 - mn0), al1 = fast_exp2(m1 - mn1);
            m0 = mn0; m1 = mn1;
            float ls0 = 0.f, ls1 = 0.f;
            uint32_t bP[2][2];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                Sc[i][0] = fast_exp2(Sc[i][0] - mn0); Sc[i][2] = fast_exp2(Sc[i][2] - mn0);
                Sc[i][1] = fast_exp2(Sc[i][1] - mn1); Sc[i][3] = fast_exp2(Sc[i][3] - mn1);
                ls0 += Sc[i][0] + Sc[i][2];
                ls1 += Sc[i][1] + Sc[i][3];
                bP[i][0] = movmatrix_trans(pack_half2(Sc[i][0], Sc[i][1]));
                bP[i][1] = movmatrix_trans(pack_half2(Sc[i][2], Sc[i][3]));
            }
            l0 = fmaf(l0, al0, ls0);
            l1 = fmaf(l1, al1, ls1);
#pragma unroll
            for (int J = 0; J < 8; ++J) { O[J][0] *= al0; O[J][2] *= al0; O[J][1] *= al1; O[J][3] *= al1; }
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            __syncwarp();
#pragma unroll
            for (int J = 0; J < 8; ++J)
#pragma unroll
                for (int kp2 = 0; kp2 < 2; ++kp2) {
                    uint32_t a[4];
                    const int blk = lane >> 3, tok = 16 * kp2 + (lane & 7) + 8 * (blk >> 1), ch = 2 * J + (blk & 1);
                    ldmatrix_x4_trans(a, vbuf + tok * 256 + ((ch ^ (tok & 7)) << 4));
                    mma16816(O[J], a[0], a[1], a[2], a[3], bP[kp2][0], bP[kp2][1]);
                }
            __syncwarp();
            if (s + 1 < n_sub) stage(vbuf, vp + (t0 + kSubTok) * kDh);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        x = seg_end;
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            l0 += __shfl_xor_sync(0xFFFFFFFFu, l0, o);
            l1 += __shfl_xor_sync(0xFFFFFFFFu, l1, o);
        }
        __syncwarp();
        float *rec = merged ? reinterpret_cast<float *>(buf) : P.partials + (size_t)(gw + tp.pair) * kPartialFloats;
        const int n0 = 2 * c, n1 = 2 * c + 1;
        if (n0 < P.G) {
            float *r0 = rec + n0 * 130;
            if (g8 == 0) { r0[0] = m0; r0[1] = l0; }
#pragma unroll
            for (int J = 0; J < 8; ++J) { r0[2 + 16 * J + g8] = O[J][0]; r0[2 + 16 * J + 8 + g8] = O[J][2]; }
        }
        if (n1 < P.G) {
            float *r1 = rec + n1 * 130;
            if (g8 == 0) { r1[0] = m1; r1[1] = l1; }
#pragma unroll
            for (int J = 0; J < 8; ++J) { r1[2 + 16 * J + g8] = O[J][1]; r1[2 + 16 * J + 8 + g8] = O[J][3]; }
        }
    }
    if (merged) {
        __syncthreads();
        const float *all = reinterpret_cast<const float *>(smem);
        const int fstride = kFp16Buf >> 2;
        float *dst = P.partials + (size_t)(blockIdx.x * W + merged_pair) * kPartialFloats;
        for (int e = tid; e < 8 * 128; e += W * 32) {
            const int n = e >> 7, dd = e & 127;
            if (n >= P.G) continue;
            float Mx = -INFINITY;
#pragma unroll
            for (int w = 0; w < W; ++w) Mx = fmaxf(Mx, all[w * fstride + n * 130]);
            float acc = 0.f, ls = 0.f;
#pragma unroll
            for (int w = 0; w < W; ++w) {
                const float *r = all + w * fstride + n * 130;
                const float f = fast_exp2(r[0] - Mx);
                acc = fmaf(r[2 + dd], f, acc);
                ls = fmaf(r[1], f, ls);
            }
            dst[n * 130 + 2 + dd] = acc;
            if (dd == 0) { dst[n * 130] = Mx; dst[n * 130 + 1] = ls; }
        }
    }
}

// ---------------------------------------------------------------- host side
constexpr int kLatencyShapedBlocks = 160;       // up to this many blocks qfold / combine run four threads per output
static int pick_warps(int buf_bytes)
{
    // measured: 12 warps at 168 registers beat 13 / 14 / 16 warps (spills, uneven schedulers)
    const int avail = 227 * 1024 - kStaticSmem;
    const int cands[3] = {12, 8, 4};
    for (int i = 0; i < 3; ++i)
        if ((size_t)cands[i] * buf_bytes <= (size_t)avail) return cands[i];
    return 0;
}
static size_t decode_smem(int W, int buf_bytes) { return kSmemHdr + (size_t)W * buf_bytes; }

size_t decode_ws_bytes(const bgtq_layout *lay, int batch, int n_layers)
{
    const size_t pairs = (size_t)n_layers * batch * lay->n_kv_heads;
    const size_t qf = pairs * kQfHalves * sizeof(__half);
    const size_t slots = (size_t)lay->sm_count * kMaxWarpsPerSM + 2 * pairs;   // warp records + one window record per pair
    return qf + slots * kPartialFloats * sizeof(float);
}

// measurement hook (bgtq_profile_decode): event pairs around the decode kernel only
static bool g_prof = false;
static std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_prof_events;
static size_t g_prof_used = 0;

void profile_decode_enable(int enable) { g_prof = enable != 0; }
int profile_decode_read(double *ms_sum, int *count)
{
    double sum = 0.0;
    for (size_t i = 0; i < g_prof_used; ++i) {
        float ms = 0.f;
        CUDA_TRY(cudaEventSynchronize(g_prof_events[i].second));
        CUDA_TRY(cudaEventElapsedTime(&ms, g_prof_events[i].first, g_prof_events[i].second));
        sum += ms;
    }
    *ms_sum = sum;
    *count = (int)g_prof_used;
    g_prof_used = 0;
    return BGTQ_OK;
}

bool profile_decode_on() { return g_prof; }
int profile_decode_begin(cudaStream_t st)
{
    if (!g_prof) return BGTQ_OK;
    if (g_prof_used == g_prof_events.size()) {
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        CUDA_TRY(cudaEventCreate(&e0));
        CUDA_TRY(cudaEventCreate(&e1));
        g_prof_events.emplace_back(e0, e1);
    }
    CUDA_TRY(cudaEventRecord(g_prof_events[g_prof_used].first, st));
    return BGTQ_OK;
}
int profile_decode_end(cudaStream_t st)
{
    if (!g_prof) return BGTQ_OK;
    CUDA_TRY(cudaEventRecord(g_prof_events[g_prof_used].second, st));
    ++g_prof_used;
    return BGTQ_OK;
}

int launch_combine(const float *partials, const int32_t *seq_len, const float *rot128, int n_layers, int batch, int Hkv, int G,
                   int64_t n_cap, int n_ctas, int W, void *out, int n_sink, int n_recent, int win_slot, bool pdl, cudaStream_t st,
                   const HeadMeta *metas, const float *rot_base)
{
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    // few blocks (a per-layer call): the latency-shaped 512-thread variant; many blocks: 128 threads
    const bool wide = n_layers * batch * Hkv * G <= kLatencyShapedBlocks;
    cfg.gridDim = dim3(n_layers * batch * Hkv * G); cfg.blockDim = dim3(wide ? 4 * kDh : kDh); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, wide ? combine_kernel<4> : combine_kernel<1>, partials, seq_len, rot128, n_layers, batch, Hkv, G, n_cap, n_ctas, W,
                       (__nv_bfloat16 *)out, n_sink, n_recent, win_slot, metas, rot_base);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

int launch_window(const void *win_k, const void *win_v, const void *q, const int32_t *seq_len, const float *rot128_t,
                  float *partials, int pairs, int batch, int Hkv, int G, int64_t n_cap, int n_sink, int n_recent,
                  float scale_log2e, int win_slot, cudaStream_t st, const HeadMeta *metas, const float *rot_t_base, bool pdl)
{
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.gridDim = dim3(pairs * G); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, window_kernel, (const __half *)win_k, (const __half *)win_v, (const __nv_bfloat16 *)q, seq_len,
                       rot128_t, partials, batch, Hkv, G, n_cap, n_sink, n_recent, scale_log2e, win_slot, metas, rot_t_base);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

template <int W, bool PAGED, bool EXACT = false, bool VG = false>
static int launch_decode_w(const DecodeParams &P, int grid, size_t smem, cudaStream_t st)
{
    if (first_use_on_device(8 + (W / 2) * 8 + (PAGED ? 1 : 0) + (EXACT ? 2 : 0) + (VG ? 4 : 0)))   // once per device, outside any stream capture
        CUDA_TRY(cudaFuncSetAttribute(decode_kernel<W, PAGED, EXACT, VG>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - kStaticSmem));
    if (int rc = profile_decode_begin(st)) return rc;
    {
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = g_prof ? 0 : 1;
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(W * 32); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, decode_kernel<W, PAGED, EXACT, VG>, P);
    }
    {
        cudaError_t le = cudaPeekAtLastError();
        if (le != cudaSuccess) {
            cudaFuncAttributes fa;
            cudaFuncGetAttributes(&fa, decode_kernel<W, PAGED, EXACT, VG>);
            set_error(std::string("decode launch: ") + cudaGetErrorString(le) + " regs=" + std::to_string(fa.numRegs) + " maxthr=" + std::to_string(fa.maxThreadsPerBlock) + " static=" + std::to_string(fa.sharedSizeBytes) + " dyn=" + std::to_string(smem) + " maxdyn=" + std::to_string(fa.maxDynamicSharedSizeBytes));
            cudaGetLastError();
            return BGTQ_ECUDA;
        }
    }
    return profile_decode_end(st);
}

int launch_decode(const bgtq_layout *lay, int layer0, int n_layers, const void *cache, const void *q,
                  const int32_t *seq_len, int batch, int64_t max_tokens, float scale, void *out,
                  void *ws, size_t, const PageMap *pm, cudaStream_t st, const Window *win)
{
    const int n_sink = win ? win->n_sink : 0, n_recent = win ? win->n_recent : 0;
    if (batch > kMaxBatch) { set_error("bgtq_decode_attention: batch > 256"); return BGTQ_EINVAL; }
    const int Hkv = lay->n_kv_heads, Hq = lay->n_q_heads, G = Hq / Hkv;
    const int64_t n_cap = (max_tokens + kTile - 1) / kTile;
    if ((double)n_layers * batch * Hkv * (double)n_cap >= 2.0e9) { set_error("bgtq_decode_attention: too many tiles for one call"); return BGTQ_EINVAL; }
    const int pairs = n_layers * batch * Hkv;
    __half *qf = reinterpret_cast<__half *>(ws);
    float *partials = reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(ws) + (size_t)pairs * kQfHalves * sizeof(__half));
    const HeadMeta *metas = lay->d_meta + (size_t)layer0 * Hkv;

    const int win_slot = win ? lay->sm_count * kMaxWarpsPerSM + pairs : -1;    // first record after the warp records
    if (win) {   // fp16 windows -> one record per (pair, query head).  Launched programmatically like qfold_kernel below (it
                 // reads the windows, q and seq_len -- complete in stream order -- and waits before it writes its record, which
                 // the previous call's combine_kernel may still read); qfold_kernel is launched programmatically behind it and
                 // the two run side by side.  Completion order: window -> qfold -> decode -> combine, each waiting for its
                 // predecessor only (qfold_kernel's wait before its first q' write also covers the previous call's decode_kernel).
        if (int rc = launch_window(win->k, win->v, q, seq_len, lay->d_rot_t + rot_offset(kDh), partials, pairs, batch, Hkv, G, n_cap,
                                   n_sink, n_recent, scale * 1.4426950408889634f, win_slot, st,
                                   lay->v_grouped ? metas : nullptr, lay->d_rot_t, !g_prof)) return rc;
    }
    const bool wideq = pairs * G <= kLatencyShapedBlocks;       // few blocks: the latency-shaped 512-thread variant
    if (!g_prof) {
        // programmatic launch: behind window_kernel (protected regime) or behind whatever precedes the call on the stream -- in
        // a layer-by-layer decode that is the previous layer's combine_kernel, which lets this kernel's prologue and dot
        // products start early (the wait sits before the first q' write).
        // A predecessor that never signals (any other kernel) just completes first, as without the attribute.
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.gridDim = dim3(pairs * G); cfg.blockDim = dim3(wideq ? 4 * kDh : kDh); cfg.dynamicSmemBytes = 0; cfg.stream = st;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, wideq ? qfold_kernel<4> : qfold_kernel<1>, metas, (const float *)lay->d_rot_t, (const __nv_bfloat16 *)q, batch, Hkv, Hq,
                           scale * 1.4426950408889634f, qf, 0, 1);
    } else if (wideq)
        qfold_kernel<4><<<pairs * G, 4 * kDh, 0, st>>>(metas, lay->d_rot_t, (const __nv_bfloat16 *)q, batch, Hkv, Hq,
                                                       scale * 1.4426950408889634f, qf, 0);
    else
        qfold_kernel<1><<<pairs * G, kDh, 0, st>>>(metas, lay->d_rot_t, (const __nv_bfloat16 *)q, batch, Hkv, Hq,
                                                   scale * 1.4426950408889634f, qf, 0);
    count_launch();
    CUDA_TRY(cudaGetLastError());

    // 128-byte aligned tile buffers; a warp's buffer also receives its partial record when the CTA merges its warps
    const int buf_bytes = (std::max(lay->max_stride, (int)(kPartialFloats * sizeof(float))) + 127) / 128 * 128;
    if (lay->sm_count + 32 >= 1024) { set_error("bgtq_decode_attention: more SMs than combine_kernel's slot list holds"); return BGTQ_EINVAL; }
    const int W = pick_warps(buf_bytes);
    if (!W) { set_error("bgtq_decode_attention: tile does not fit shared memory"); return BGTQ_EINVAL; }
    DecodeParams P;
    P.metas = metas; P.cache = (const uint8_t *)cache; P.qf = qf; P.seq_len = seq_len; P.cb16 = lay->d_cb16;
    P.hcb16 = lay->cb_exact ? lay->d_hcb16 + (size_t)layer0 * Hkv * 2 * kHeadLutHalves : nullptr;
    P.partials = partials; P.n_cap = n_cap; P.n_layers = n_layers; P.batch = batch; P.Hkv = Hkv; P.G = G;
    P.buf_bytes = buf_bytes;
    P.pages = pm ? pm->table : nullptr; P.pstride = pm ? pm->table_stride : 0; P.n_pages = pm ? pm->n_pages : 0;
    P.n_sink = n_sink; P.n_recent = n_recent;
    const int grid = lay->sm_count;
    const size_t smem = decode_smem(W, buf_bytes);
    int rc;
    if (lay->v_grouped) {
        if (pm) { set_error("bgtq_decode_attention_paged: not built for V-side groups"); return BGTQ_EINVAL; }
        if (lay->cb_exact)
            switch (W) {
            case 12: rc = launch_decode_w<12, false, true, true>(P, grid, smem, st); break;
            case 8: rc = launch_decode_w<8, false, true, true>(P, grid, smem, st); break;
            default: rc = launch_decode_w<4, false, true, true>(P, grid, smem, st); break;
            }
        else
            switch (W) {
            case 12: rc = launch_decode_w<12, false, false, true>(P, grid, smem, st); break;
            case 8: rc = launch_decode_w<8, false, false, true>(P, grid, smem, st); break;
            default: rc = launch_decode_w<4, false, false, true>(P, grid, smem, st); break;
            }
    } else if (lay->cb_exact) {
        if (pm) { set_error("bgtq_decode_attention_paged: not built for exact-density codebooks"); return BGTQ_EINVAL; }
        switch (W) {
        case 12: rc = launch_decode_w<12, false, true>(P, grid, smem, st); break;
        case 8: rc = launch_decode_w<8, false, true>(P, grid, smem, st); break;
        default: rc = launch_decode_w<4, false, true>(P, grid, smem, st); break;
        }
    } else if (pm) {
        switch (W) {
        case 12: rc = launch_decode_w<12, true>(P, grid, smem, st); break;
        case 8: rc = launch_decode_w<8, true>(P, grid, smem, st); break;
        default: rc = launch_decode_w<4, true>(P, grid, smem, st); break;
        }
    } else {
        switch (W) {
        case 12: rc = launch_decode_w<12, false>(P, grid, smem, st); break;
        case 8: rc = launch_decode_w<8, false>(P, grid, smem, st); break;
        default: rc = launch_decode_w<4, false>(P, grid, smem, st); break;
        }
    }
    if (rc != BGTQ_OK) return rc;
    count_launch();
    CUDA_TRY(cudaGetLastError());

    return launch_combine(partials, seq_len, lay->d_rot + rot_offset(kDh), n_layers, batch, Hkv, G, n_cap, grid, W, out, n_sink,
                          n_recent, win_slot, !g_prof, st, lay->v_grouped ? metas : nullptr, lay->d_rot);
}

int launch_window_append(const void *k_new, const void *v_new, int dt, int n_layers, int batch, int n_new, int Hkv,
                         const int32_t *seq_len, int64_t max_tokens, void *win_k, void *win_v, int n_sink, int n_recent, cudaStream_t st)
{
    const int grid = n_layers * batch * n_new;
    if (dt == BGTQ_F32)
        window_append_kernel<float><<<grid, 128, 0, st>>>((const float *)k_new, (const float *)v_new, seq_len, (__half *)win_k,
                                                          (__half *)win_v, batch, n_new, Hkv, n_sink, n_recent, max_tokens);
    else
        window_append_kernel<__nv_bfloat16><<<grid, 128, 0, st>>>((const __nv_bfloat16 *)k_new, (const __nv_bfloat16 *)v_new, seq_len,
                                                                  (__half *)win_k, (__half *)win_v, batch, n_new, Hkv, n_sink, n_recent, max_tokens);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

// ---------------------------------------------------------------- host side of the fp16 comparison path
size_t fp16_ws_bytes(int sm_count, int batch, int n_layers, int Hkv)
{
    return ((size_t)sm_count * kMaxWarpsPerSM + (size_t)n_layers * batch * Hkv) * kPartialFloats * sizeof(float);
}

int launch_fp16_decode(int n_layers, int batch, int Hq, int Hkv, const void *k_cache, const void *v_cache,
                       const void *q, const int32_t *seq_len, int64_t max_tokens, float scale, void *out,
                       void *ws, size_t ws_bytes, cudaStream_t st)
{
    static int sm_count = 0;
    if (!sm_count) {
        int dev = 0;
        CUDA_TRY(cudaGetDevice(&dev));
        CUDA_TRY(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    }
    if (batch > kMaxBatch) { set_error("bgtq_fp16_decode_attention: batch > 256"); return BGTQ_EINVAL; }
    if (ws_bytes < fp16_ws_bytes(sm_count, batch, n_layers, Hkv)) { set_error("bgtq_fp16_decode_attention: workspace too small"); return BGTQ_EWORKSPACE; }
    const size_t smem = (size_t)kFp16Warps * kFp16Buf;
    if (first_use_on_device(2)) {
        CUDA_TRY(cudaFuncSetAttribute(fp16_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    Fp16Params P;
    P.k_cache = (const __half *)k_cache; P.v_cache = (const __half *)v_cache; P.q = (const __nv_bfloat16 *)q;
    P.seq_len = seq_len; P.partials = (float *)ws; P.n_cap = (max_tokens + kTile - 1) / kTile;
    P.n_layers = n_layers; P.batch = batch; P.Hkv = Hkv; P.G = Hq / Hkv; P.scale_log2e = scale * 1.4426950408889634f;
    fp16_decode_kernel<<<sm_count, kFp16Warps * 32, smem, st>>>(P);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    combine_kernel<1><<<n_layers * batch * Hkv * P.G, kDh, 0, st>>>(P.partials, seq_len, nullptr, n_layers, batch, Hkv, P.G,
                                                                 P.n_cap, sm_count, kFp16Warps, (__nv_bfloat16 *)out, 0, 0, -1,
                                                                    (const HeadMeta *)nullptr, (const float *)nullptr);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

// ---------------------------------------------------------------- NEXT #1: prefill attention over the packed cache
// "each program owns a tile of queries, streams the compressed K/V tiles, decodes them into
// kernel-local temporaries ... and accumulates under a causal mask with an online softmax".  First cut: a CTA owns
// 16*(8/G) query tokens x the G query heads of one KV head; every 128-token packed tile is staged by one TMA bulk
// copy, unpacked ONCE by all 8 warps into shared memory as fp16 (K^ with its group norms, in grouped coordinate
// order; V^T with its token norms, both in the rotated domain), and then consumed FlashAttention-2 style with
// ldmatrix + mma.sync by the 8 warps (16 query rows each).  The rotation stays folded: queries arrive as q'
// (plain layout of qfold_kernel), the output is de-rotated by derotate_kernel.  The unpack is amortised over 128
// query rows, so this kernel is bound by the (legacy) tensor path, not by the ALU unpack.
struct PrefillParams {
    const HeadMeta *metas;      // [Hkv] of the layer
    const uint8_t *cache;
    const __half *qp;           // q' plain: [batch*n_q][Hkv][8][128]
    const int32_t *seq_len;
    const uint16_t *cb16;
    float *opart;               // [batch*n_q][Hq][128] fp32, rotated domain, normalised
    int64_t n_cap;
    int batch, n_q, Hkv, G, raw_bytes;
};

struct PUnit { int off, b, nc, ustart, group; };

// Shared-memory layouts of the unpacked fp16 tiles [row][k] (row = token for K^, dim for V^T):
//   UMMA = false: 256-byte rows, 16-byte chunks XOR-swizzled with (row & 7)              (ldmatrix path)
//   UMMA = true : the tcgen05 K-major SWIZZLE_128B operand layout: two [128 x 64] blocks of 16 KB, 128-byte rows,
//                 chunk ^ (row & 7); 8-row groups 1024 B apart (the SBO of the descriptor)
template <bool UMMA>
__device__ __forceinline__ int tile_off(int row, int k)
{
    if (UMMA) return (k >> 6) * 16384 + row * 128 + (((((k & 63) >> 3) ^ (row & 7)) << 4) | ((k & 7) << 1));
    return row * 256 + ((((k >> 3) ^ (row & 7)) << 4) | ((k & 7) << 1));
}

template <int B, bool UMMA = false>
__device__ __forceinline__ void prefill_decode_k(const uint32_t *raw, const PUnit &U, int lane, const uint32_t *pools,
                                                 const uint16_t *lut, const __half *kn, unsigned char *khat)
{
    const int g8 = lane >> 2, c = lane & 3;
    uint32_t w[B], h[16];
    if (U.nc == 4) load_unit_full<B>(raw + (U.off >> 2), lane, w);
    else load_unit_partial<B>(raw + (U.off >> 2), g8, c, U.nc, w);
    decode_unit<B, true>(w, pools, lut, h);
    if (c < U.nc) {
        const int col = U.ustart + 2 * c;
        if (UMMA) {
            // the norm row of a group is stored so that the 16 tokens of a lane (16 i + 8 p + g8) are 16 consecutive fp16:
            // `kn` points at the raw row of the unit's group
            const uint4 *np = reinterpret_cast<const uint4 *>(kn + g8 * 16);
            const uint4 n0 = np[0], n1 = np[1];
            const uint32_t nw[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    const int tok = 16 * i + 8 * p + g8;
                    // (h, h) * (n, n): the half of the norm pair is broadcast by the multiply's operand select, not by a PRMT
                    const __half2 nn = *reinterpret_cast<const __half2 *>(&nw[i]);
                    const __half2 pr = __hmul2(*reinterpret_cast<const __half2 *>(&h[2 * i + p]), p ? __high2half2(nn) : __low2half2(nn));
                    *reinterpret_cast<uint32_t *>(khat + tile_off<UMMA>(tok, col)) = *reinterpret_cast<const uint32_t *>(&pr);
                }
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    const int tok = 16 * i + 8 * p + g8;
                    const uint32_t n2 = (uint32_t)__half_as_ushort(kn[U.group * 128 + tok]) * 0x10001u;
                    const uint32_t v = hmul2_u(h[2 * i + p], n2);
                    *reinterpret_cast<uint32_t *>(khat + tile_off<UMMA>(tok, col)) = v;
                }
        }
    }
}

template <int B, bool UMMA = false>
__device__ __forceinline__ void prefill_decode_v(const uint32_t *vcodes, int J, int lane, const uint32_t *pools,
                                                 const uint16_t *lut, const __half *vn, unsigned char *vhat_t, int only_rho = -1)
{
    const int gq = lane >> 2, c = lane & 3;
#pragma unroll
    for (int rho = 0; rho < 2; ++rho) {
        if (only_rho >= 0 && rho != only_rho) continue;
        uint32_t w[B], h[16];
        load_unit_full<B>(vcodes + (2 * J + rho) * 32 * B, lane, w);
        decode_unit<B, true>(w, pools, lut, h);
        const int dim = 16 * J + 8 * rho + gq;
#pragma unroll
        for (int kp = 0; kp < 8; ++kp)
#pragma unroll
            for (int o = 0; o < 2; ++o) {
                const int tok = 16 * kp + 8 * o + 2 * c;                   // tokens tok, tok+1
                const uint32_t n2 = *reinterpret_cast<const uint32_t *>(vn + tok);
                const uint32_t v = hmul2_u(h[2 * kp + o], n2);
                *reinterpret_cast<uint32_t *>(vhat_t + tile_off<UMMA>(dim, tok)) = v;
            }
    }
}

// ---------------------------------------------------------------- prefill on the 5th-generation tensor cores
// Same problem and interface as prefill_kernel, but both contractions run as tcgen05.mma (kind::f16, fp32 accumulators in
// tensor memory), issued by one thread.  A CTA owns 128 query rows (128/G tokens x G heads of one KV head):
//   shared memory: Q' [128 rows x 128 coords], K^ [128 tokens x 128 coords], V^T [128 dims x 128 tokens] and
//                  P [128 rows x 128 tokens], all fp16 in the K-major SWIZZLE_128B operand layout (two 16 KB blocks each),
//                  + the raw packed tile (TMA bulk copy);
//   tensor memory: S = Q' K^T in columns [0,128), O in columns [128,256); row r of S / O is TMEM lane r.
// Per 128-token tile: all 8 warps unpack K^ -> S MMA (async) -> unpack V^T while it runs -> softmax straight out of TMEM
// (thread = one row x 32 columns: no shuffles; the four column quarters meet through shared memory) -> P to shared memory,
// O rescaled in TMEM when a row maximum moved -> PV MMA (async), which overlaps the next tile's K^ unpack.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr)
{
    // K-major SWIZZLE_128B shared-memory operand: start address >> 4 in bits [0,14); leading byte offset (not used by
    // swizzled K-major layouts) = 1 in [16,30); stride byte offset = 1024 B (8 rows x 128 B) >> 4 in [32,46);
    // descriptor version 1 (sm_100) in [46,48); layout type 2 = SWIZZLE_128B in [61,64)
    return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void umma_f16_ss(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
// D[128 x 128] (+)= A[128 x 128] . B[128 x 128]^T; each operand = two K blocks of [128 x 64] fp16, 16 KB apart
__device__ __forceinline__ void umma_128x128x128(uint32_t d_tmem, uint32_t a_s, uint32_t b_s, bool accumulate)
{
    // instruction descriptor: D format f32 (1) in [4,6); A, B format f16 (0); both K-major; N >> 3 in [17,23); M >> 4 in [24,29)
    constexpr uint32_t idesc = (1u << 4) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
#pragma unroll
    for (int kb = 0; kb < 2; ++kb)
#pragma unroll
        for (int k = 0; k < 4; ++k)                          // UMMA_K = 16 fp16 = 32 bytes inside the 128-byte swizzle row
            umma_f16_ss(d_tmem, umma_desc_sw128(a_s + kb * 16384 + k * 32), umma_desc_sw128(b_s + kb * 16384 + k * 32), idesc,
                        (accumulate || kb || k) ? 1u : 0u);
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
                 :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
}
__device__ __forceinline__ float fmax3(float a, float b, float c)
{
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));     // FMNMX3 (sm_100)
    return r;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

constexpr int kTcThreads = 512;                       // 16 warps: 4 per TMEM lane quadrant
__host__ __device__ constexpr int tc_operand_bytes(int RT) { return RT * 32768 + 32768 + 32768 + RT * 32768; }   // Q', K^, V^T, P

// RT = 128-row query tiles per CTA (1 or 2).  With RT = 2 one unpack of a packed tile serves 256 query rows
// (32 tokens x 8 heads at G = 8): S0, S1 in TMEM columns [0,256), O0, O1 in [256,512) -- the whole tensor memory --
// and 192 KB of operands in shared memory, so it is used whenever the raw tile still fits beside them.
template <int RT>
__global__ void __launch_bounds__(kTcThreads, 1)
prefill_tc_kernel(const PrefillParams P)
{
    constexpr int NG = 4 / RT;                        // column groups per row: each thread owns 128 / NG columns of one row
    constexpr int NCH = RT;                           // ... i.e. NCH chunks of 32 columns
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(16) uint16_t lut[kLutHalves];
    __shared__ uint32_t pools[16];
    __shared__ __align__(8) uint64_t bars[3];         // raw tile landed / S ready / PV done
    __shared__ PUnit units[2 * kMaxKSteps];
    __shared__ int n_units_s;
    __shared__ uint32_t tmem_base_s;
    __shared__ float rmax[NG][RT * 128], rsum[NG][RT * 128];
    __shared__ __align__(16) __half vn[128];
    unsigned char *qs = smem, *khat = smem + RT * 32768, *vhat_t = khat + 32768, *ps = vhat_t + 32768;
    uint32_t *raw = reinterpret_cast<uint32_t *>(smem + tc_operand_bytes(RT));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int h = blockIdx.y, b = blockIdx.z, G = P.G;
    const HeadMeta &M = P.metas[h];
    const int TQ = RT * 128 / G;
    int64_t slen = P.seq_len[b];
    slen = slen > P.n_cap * kTile ? P.n_cap * kTile : slen;
    const int i_first = blockIdx.x * TQ;
    const int i_last = min(P.n_q, i_first + TQ) - 1;
    const int64_t pos0 = slen - P.n_q;                              // position of query token 0
    if (i_first >= P.n_q || pos0 < 0) return;
    const int n_tiles = (int)((pos0 + i_last) / kTile) + 1;

    build_lut(P.cb16, lut, tid, kTcThreads, true);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "n"(RT * 256) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int i = tid; i < (32768 + 32768) / 16; i += kTcThreads) reinterpret_cast<uint4 *>(khat)[i] = make_uint4(0, 0, 0, 0);   // K^ (zero-width blocks stay 0), V^T
    const uint32_t bar_raw = smem_u32(&bars[0]), bar_s = smem_u32(&bars[1]), bar_o = smem_u32(&bars[2]);
    if (tid == 0) {
        int nu = 0, j = 0;
        for (int ks = 0; ks < M.n_ksteps; ++ks) {
            const KStep &K = M.ksteps[ks];
            const int g = K.flags >> 4;
            if (K.flags & 1) j = 0;
            units[nu++] = PUnit{K.off0, K.b, K.nc0, M.gstart[g] + 8 * j, g};
            ++j;
            if (K.off1 != 0xFFFF) { units[nu++] = PUnit{K.off1, K.b, K.nc1, M.gstart[g] + 8 * j, g}; ++j; }
        }
        n_units_s = nu;
        mbar_init(bar_raw, 1);
        mbar_init(bar_s, 1);
        mbar_init(bar_o, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    {   // Q' rows -> the A operands.  Row r of the CTA = (token r / G, head r % G); rows past n_q are zero.
        constexpr int TPR = 4 / RT, NV = 4 * RT;                    // threads per row, 16-byte vectors per thread
        const int r = tid / TPR, part = tid % TPR;
        const int kb = (part * 8 * NV) >> 6, j0 = ((part * 8 * NV) & 63) >> 3;
        const int ti = i_first + r / G, n = r % G, rr = r & 127;
        const bool valid = ti < P.n_q;
        const uint4 *src = reinterpret_cast<const uint4 *>(P.qp + ((((size_t)b * P.n_q + (valid ? ti : 0)) * P.Hkv + h) * 8 + n) * kDh + part * 8 * NV);
#pragma unroll
        for (int jj = 0; jj < NV; ++jj) {
            const uint4 v = valid ? __ldg(src + jj) : make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4 *>(qs + (r >> 7) * 32768 + kb * 16384 + rr * 128 + (((j0 + jj) ^ (rr & 7)) << 4)) = v;
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = tmem_base_s;
    if (tid == 0) build_pools(lut, pools);
    __syncthreads();                                                // pools are read by the first unpack
    const int n_units = n_units_s, b_v = M.b_v;
    const uint8_t *region = P.cache + P.n_cap * ((int64_t)P.batch * M.layer_prefix + (int64_t)b * M.layer_sum + M.head_prefix);
    const uint32_t raw_s = smem_u32(raw);
    if (tid == 0) { mbar_expect_tx(bar_raw, M.tile_stride); bulk_g2s(raw_s, region, M.tile_stride, bar_raw); }

    // softmax ownership: TMEM lane quadrant = warp & 3 (a warp can only touch its own quadrant); the 4 warps of a quadrant
    // split into RT row tiles x NG column groups
    const int quad = warp & 3, rt = (warp >> 2) % RT, cg = (warp >> 2) / RT;
    const int row = 32 * quad + lane, crow = rt * 128 + row, c_lo = cg * (128 / NG);
    const int64_t prow = pos0 + i_first + crow / G;                 // position of this row's query token
    const uint32_t t_s = tm + ((uint32_t)(32 * quad) << 16) + (uint32_t)(rt * 128 + c_lo), t_o = t_s + RT * 128u;
    const uint32_t qs_s = smem_u32(qs), khat_s = smem_u32(khat), vhat_s = smem_u32(vhat_t), ps_s = smem_u32(ps);
    unsigned char *prow_s = ps + rt * 32768 + row * 128;
    float m_run = -INFINITY, l_run = 0.f;
    uint32_t ph_raw = 0, ph_s = 0, ph_o = 0;

    for (int t = 0; t < n_tiles; ++t) {
        // ---- a. raw tile t landed: linearise the norms, unpack K^ (its buffer is free: S(t-1) was waited for), start S
        mbar_wait(bar_raw, ph_raw);
        ph_raw ^= 1;
        if (tid < 128)      // V norms in token order for the V^T unpack (K norms are read from the raw rows directly)
            vn[tid] = reinterpret_cast<const __half *>(reinterpret_cast<const unsigned char *>(raw) + M.vnorm_off)[(tid & 7) * 16 + (tid >> 4) * 2 + ((tid >> 3) & 1)];
        for (int u = warp; u < n_units; u += kTcThreads / 32) {
            const PUnit U = units[u];
            const __half *kn = reinterpret_cast<const __half *>(reinterpret_cast<const unsigned char *>(raw) + M.knorm_off + 256 * U.group);
            switch (U.b) {
            case 1: prefill_decode_k<1, true>(raw, U, lane, pools, lut, kn, khat); break;
            case 2: prefill_decode_k<2, true>(raw, U, lane, pools, lut, kn, khat); break;
            case 3: prefill_decode_k<3, true>(raw, U, lane, pools, lut, kn, khat); break;
            case 4: prefill_decode_k<4, true>(raw, U, lane, pools, lut, kn, khat); break;
            case 5: prefill_decode_k<5, true>(raw, U, lane, pools, lut, kn, khat); break;
            case 6: prefill_decode_k<6, true>(raw, U, lane, pools, lut, kn, khat); break;
            case 7: prefill_decode_k<7, true>(raw, U, lane, pools, lut, kn, khat); break;
            default: prefill_decode_k<8, true>(raw, U, lane, pools, lut, kn, khat); break;
            }
        }
        fence_proxy_async();                                         // generic-proxy writes of Q', K^ -> visible to the MMA
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
#pragma unroll
            for (int r = 0; r < RT; ++r) umma_128x128x128(tm + r * 128, qs_s + r * 32768, khat_s, false);   // S_r = Q'_r . K^T
            umma_commit(bar_s);
        }
        // ---- b. unpack V^T while S runs (its buffer and P are free once PV(t-1) has completed)
        if (t > 0) {
            mbar_wait(bar_o, ph_o);
            ph_o ^= 1;
            tc_fence_after();
        }
        {
            const uint32_t *vcodes = raw + (M.vcode_off >> 2);
            switch (b_v) {
            case 1: prefill_decode_v<1, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            case 2: prefill_decode_v<2, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            case 3: prefill_decode_v<3, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            case 4: prefill_decode_v<4, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            case 5: prefill_decode_v<5, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            case 6: prefill_decode_v<6, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            case 7: prefill_decode_v<7, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            default: prefill_decode_v<8, true>(vcodes, warp >> 1, lane, pools, lut, vn, vhat_t, warp & 1); break;
            }
        }
        // ---- c. softmax of this thread's row x (128 / NG) columns, straight from tensor memory (log2 domain), in two
        //      passes over TMEM (maximum, then exponentials) so that no more than 32 logits are in registers at a time
        mbar_wait(bar_s, ph_s);
        ph_s ^= 1;
        tc_fence_after();
        const int rel = (int)max((int64_t)-1, min((int64_t)1 << 20, prow - ((int64_t)t * kTile + c_lo)));   // columns > rel are in the future
        // (all but the last one or two tiles of a row are fully visible: warp-uniform fast path without the mask)
        const bool nomask = __all_sync(0xFFFFFFFFu, rel >= 128 / NG - 1);
        float mx = -INFINITY;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            uint32_t sr[32];
            tmem_ld32(t_s + 32 * ch, sr);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (nomask) {
#pragma unroll
                for (int i = 0; i < 32; i += 2) mx = fmax3(mx, __uint_as_float(sr[i]), __uint_as_float(sr[i + 1]));
            } else {
#pragma unroll
                for (int i = 0; i < 32; ++i) mx = fmaxf(mx, 32 * ch + i > rel ? -INFINITY : __uint_as_float(sr[i]));
            }
        }
        rmax[cg][crow] = mx;
        __syncthreads();                                             // (also: every warp is done with the raw tile)
        if (tid == 0 && t + 1 < n_tiles) {
            fence_proxy_async();
            mbar_expect_tx(bar_raw, M.tile_stride);
            bulk_g2s(raw_s, region + (int64_t)(t + 1) * M.tile_stride, M.tile_stride, bar_raw);
        }
        float mn = m_run;                                            // finite after tile 0: it holds position 0
#pragma unroll
        for (int g2 = 0; g2 < NG; ++g2) mn = fmaxf(mn, rmax[g2][crow]);
        const float alpha = fast_exp2(m_run - mn);
        m_run = mn;
        float ls = 0.f;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            uint32_t sr[32];
            tmem_ld32(t_s + 32 * ch, sr);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int j = 0; j < 4; ++j) {                            // 8 tokens = one 16-byte chunk of the P row
                float p[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int i = 32 * ch + 8 * j + e;
                    p[e] = (!nomask && i > rel) ? 0.f : fast_exp2(__uint_as_float(sr[8 * j + e]) - mn);
                    ls += p[e];
                }
                const uint4 v = make_uint4(pack_half2(p[0], p[1]), pack_half2(p[2], p[3]), pack_half2(p[4], p[5]), pack_half2(p[6], p[7]));
                const int col = c_lo + 32 * ch + 8 * j;              // token column of the chunk: K block col >> 6, chunk (col & 63) >> 3
                *reinterpret_cast<uint4 *>(prow_s + (col >> 6) * 16384 + ((((col & 63) >> 3) ^ (row & 7)) << 4)) = v;
            }
        }
        l_run = fmaf(l_run, alpha, ls);
        if (t > 0 && __any_sync(0xFFFFFFFFu, alpha != 1.f)) {        // a row maximum moved: rescale O in place
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                uint32_t o[32];
                tmem_ld32(t_o + 32 * ch, o);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                tmem_st32(t_o + 32 * ch, o);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
        fence_proxy_async();                                         // P, V^T -> visible to the MMA
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
#pragma unroll
            for (int r = 0; r < RT; ++r) umma_128x128x128(tm + (RT + r) * 128, ps_s + r * 32768, vhat_s, t > 0);   // O_r (+)= P_r . V^
            umma_commit(bar_o);
        }
    }
    // ---- normalise and store the rotated-domain output rows (fp32); derotate_kernel finishes them
    mbar_wait(bar_o, ph_o);
    tc_fence_after();
    rsum[cg][crow] = l_run;
    __syncthreads();
    float lt = 0.f;
#pragma unroll
    for (int g2 = 0; g2 < NG; ++g2) lt += rsum[g2][crow];
    const float inv = 1.f / lt;
    const int ti = i_first + crow / G, n = crow % G;
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        uint32_t o[32];
        tmem_ld32(t_o + 32 * ch, o);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (ti < P.n_q) {
            float4 *dst = reinterpret_cast<float4 *>(P.opart + (((size_t)b * P.n_q + ti) * (P.Hkv * G) + h * G + n) * kDh + c_lo + 32 * ch);
#pragma unroll
            for (int i = 0; i < 8; ++i)
                dst[i] = make_float4(__uint_as_float(o[4 * i]) * inv, __uint_as_float(o[4 * i + 1]) * inv,
                                     __uint_as_float(o[4 * i + 2]) * inv, __uint_as_float(o[4 * i + 3]) * inv);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tm), "n"(RT * 256) : "memory");
}

// ---------------------------------------------------------------- prefill, warp-specialised (two 128-row query tiles per CTA)
// Same operands, tensor-memory map and arithmetic as prefill_tc_kernel<2>, but the three kinds of work run concurrently
// on different warps and different pipes instead of in block-wide phases:
//   warps 0-7   softmax: TMEM lane quadrant = warp & 3, query tile = warp >> 2; a thread owns one whole row (128 logits):
//               no exchange between threads at all; MUFU-bound
//   warps 8-14  producers: unpack K^ / V^T of the next tile into the operand buffers (ALU-pipe bound)
//   warp 15     one thread issues the TMA bulk copies of the packed half tiles and the tcgen05.mma groups
// and hand over through mbarriers (one completion per tile each; a waiter uses the parity of the tile index):
//   kfull/vfull  TMA: [K codes|K norms] / [V norms|V codes] of tile t landed
//   kready/vready  7 producer warps: K^ / V^T(t) written (the raw half is free again)
//   sfull        tcgen05.commit: S(t) = Q' K^T complete (K^ is free again)
//   sfree        8 softmax warps: S(t) has been read (S(t+1) may overwrite it)
//   pready       8 softmax warps: P(t) written, O rescaled
//   odone        tcgen05.commit: O += P(t) V^(t) complete (V^T and P are free again, O is stable)
enum { WS_KFULL = 0, WS_VFULL, WS_KREADY, WS_VREADY, WS_SFULL, WS_SFREE, WS_PREADY, WS_ODONE, WS_NBARS };
#ifndef BGTQ_WS_PRODUCERS
#define BGTQ_WS_PRODUCERS 11
#endif
constexpr int kWsProducers = BGTQ_WS_PRODUCERS;     // unpack warps (they are the critical path: 7 were busy 87 % of the time)
constexpr int kWsThreads = 32 * (8 + kWsProducers + 1);   // 8 softmax warps, the producers, one issuer warp


__global__ void __launch_bounds__(kWsThreads, 1)
prefill_ws_kernel(const PrefillParams P)
{
    constexpr int RT = 2;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(16) uint16_t lut[kLutHalves];
    __shared__ uint32_t pools[16];
    __shared__ __align__(8) uint64_t bars[WS_NBARS];
    __shared__ PUnit units[2 * kMaxKSteps];
    __shared__ int n_units_s;
    __shared__ uint32_t tmem_base_s;
    __shared__ __align__(16) __half vn_w[kWsProducers][128];        // V norms in token order, one private copy per producer warp
    unsigned char *qs = smem, *khat = smem + RT * 32768, *vhat_t = khat + 32768, *ps = vhat_t + 32768;
    uint32_t *raw = reinterpret_cast<uint32_t *>(smem + tc_operand_bytes(RT));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int h = blockIdx.y, b = blockIdx.z, G = P.G;
    const HeadMeta &M = P.metas[h];
    const int TQ = RT * 128 / G;
    int64_t slen = P.seq_len[b];
    slen = slen > P.n_cap * kTile ? P.n_cap * kTile : slen;
    const int i_first = blockIdx.x * TQ;
    const int i_last = min(P.n_q, i_first + TQ) - 1;
    const int64_t pos0 = slen - P.n_q;                              // position of query token 0
    if (i_first >= P.n_q || pos0 < 0) return;
    const int n_tiles = (int)((pos0 + i_last) / kTile) + 1;

    build_lut(P.cb16, lut, tid, kWsThreads, true);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" :: "r"(smem_u32(&tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int i = tid; i < (32768 + 32768) / 16; i += kWsThreads) reinterpret_cast<uint4 *>(khat)[i] = make_uint4(0, 0, 0, 0);   // K^ (zero-width blocks stay 0), V^T
    uint32_t bar[WS_NBARS];
#pragma unroll
    for (int i = 0; i < WS_NBARS; ++i) bar[i] = smem_u32(&bars[i]);
    if (tid == 0) {
        int nu = 0, j = 0;
        for (int ks = 0; ks < M.n_ksteps; ++ks) {
            const KStep &K = M.ksteps[ks];
            const int g = K.flags >> 4;
            if (K.flags & 1) j = 0;
            units[nu++] = PUnit{K.off0, K.b, K.nc0, M.gstart[g] + 8 * j, g};
            ++j;
            if (K.off1 != 0xFFFF) { units[nu++] = PUnit{K.off1, K.b, K.nc1, M.gstart[g] + 8 * j, g}; ++j; }
        }
        n_units_s = nu;
        mbar_init(bar[WS_KFULL], 1);
        mbar_init(bar[WS_VFULL], 1);
        mbar_init(bar[WS_KREADY], kWsProducers);
        mbar_init(bar[WS_VREADY], kWsProducers);
        mbar_init(bar[WS_SFULL], 1);
        mbar_init(bar[WS_SFREE], 8);
        mbar_init(bar[WS_PREADY], 8);
        mbar_init(bar[WS_ODONE], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    if (tid < 512) {   // Q' rows -> the A operands.  Row r of the CTA = (token r / G, head r % G); rows past n_q are zero.
        constexpr int TPR = 4 / RT, NV = 4 * RT;                    // threads per row, 16-byte vectors per thread
        const int r = tid / TPR, part = tid % TPR;
        const int kb = (part * 8 * NV) >> 6, j0 = ((part * 8 * NV) & 63) >> 3;
        const int ti = i_first + r / G, n = r % G, rr = r & 127;
        const bool valid = ti < P.n_q;
        const uint4 *src = reinterpret_cast<const uint4 *>(P.qp + ((((size_t)b * P.n_q + (valid ? ti : 0)) * P.Hkv + h) * 8 + n) * kDh + part * 8 * NV);
#pragma unroll
        for (int jj = 0; jj < NV; ++jj) {
            const uint4 v = valid ? __ldg(src + jj) : make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4 *>(qs + (r >> 7) * 32768 + kb * 16384 + rr * 128 + (((j0 + jj) ^ (rr & 7)) << 4)) = v;
        }
    }
    fence_proxy_async();                                            // Q', zero fill -> visible to the MMA
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = tmem_base_s;
    if (tid == 0) build_pools(lut, pools);
    __syncthreads();
    const int n_units = n_units_s, b_v = M.b_v;
    const uint8_t *region = P.cache + P.n_cap * ((int64_t)P.batch * M.layer_prefix + (int64_t)b * M.layer_sum + M.head_prefix);
    const uint32_t raw_s = smem_u32(raw), kbytes = M.vnorm_off, vbytes = M.tile_stride - M.vnorm_off;
    const uint32_t qs_s = smem_u32(qs), khat_s = smem_u32(khat), vhat_s = smem_u32(vhat_t), ps_s = smem_u32(ps);

    if (warp == 8 + kWsProducers) {
        // ================= issuer: TMA + tcgen05.mma, one thread
        if (lane == 0) {
            mbar_expect_tx(bar[WS_KFULL], kbytes); bulk_g2s(raw_s, region, kbytes, bar[WS_KFULL]);
            mbar_expect_tx(bar[WS_VFULL], vbytes); bulk_g2s(raw_s + kbytes, region + kbytes, vbytes, bar[WS_VFULL]);
            // Issue order S(0), [S(t+1), O(t)] for t = 0 ..: S(t+1) = Q'K^T of the NEXT tile goes to the tensor pipe ahead of
            // O(t) += P(t) V^(t), so the softmax warps get S(t+1) one MMA sooner (the S buffer is free as soon as softmax(t) has
            // read it, which is just before P(t) is ready).
            auto issue_s = [&](int t) {
                mbar_wait(bar[WS_KREADY], t & 1);
                if (t > 0) mbar_wait(bar[WS_SFREE], (t - 1) & 1);
                tc_fence_after();
#pragma unroll
                for (int r = 0; r < RT; ++r) umma_128x128x128(tm + r * 128, qs_s + r * 32768, khat_s, false);          // S_r = Q'_r . K^T
                umma_commit(bar[WS_SFULL]);
                if (t + 1 < n_tiles) {                               // the producers are done with the raw K half
                    const uint8_t *src = region + (int64_t)(t + 1) * M.tile_stride;
                    mbar_expect_tx(bar[WS_KFULL], kbytes); bulk_g2s(raw_s, src, kbytes, bar[WS_KFULL]);
                }
            };
            issue_s(0);
            for (int t = 0; t < n_tiles; ++t) {
                const uint32_t par = t & 1;
                // whichever is ready first; S(t+1) ahead of O(t) when both are
                bool s_done = t + 1 >= n_tiles, v_req = t + 1 >= n_tiles;
                for (;;) {
                    if (!s_done && mbar_test(bar[WS_KREADY], (t + 1) & 1) && mbar_test(bar[WS_SFREE], par)) { issue_s(t + 1); s_done = true; }
                    const bool vr = mbar_test(bar[WS_VREADY], par);
                    if (vr && !v_req) {                              // the producers are done with the raw V half: fetch the next one now
                        const uint8_t *src = region + (int64_t)(t + 1) * M.tile_stride + kbytes;
                        mbar_expect_tx(bar[WS_VFULL], vbytes); bulk_g2s(raw_s + kbytes, src, vbytes, bar[WS_VFULL]);
                        v_req = true;
                    }
                    if (vr && mbar_test(bar[WS_PREADY], par)) break;
                }
                tc_fence_after();
#pragma unroll
                for (int r = 0; r < RT; ++r) umma_128x128x128(tm + (RT + r) * 128, ps_s + r * 32768, vhat_s, t > 0);   // O_r (+)= P_r . V^
                umma_commit(bar[WS_ODONE]);
                if (!s_done) issue_s(t + 1);
            }
        }
    } else if (warp >= 8) {
        // ================= producers: unpack K^ and V^T of every tile
        const int pw = warp - 8;
        __half *vn = vn_w[pw];
        for (int t = 0; t < n_tiles; ++t) {
            const uint32_t par = t & 1, parp = (t - 1) & 1;
            mbar_wait(bar[WS_KFULL], par);
            if (t > 0) mbar_wait(bar[WS_SFULL], parp);               // S(t-1) has consumed K^
            for (int u = pw; u < n_units; u += kWsProducers) {
                const PUnit U = units[u];
                const __half *kn = reinterpret_cast<const __half *>(reinterpret_cast<const unsigned char *>(raw) + M.knorm_off + 256 * U.group);
                switch (U.b) {
                case 1: prefill_decode_k<1, true>(raw, U, lane, pools, lut, kn, khat); break;
                case 2: prefill_decode_k<2, true>(raw, U, lane, pools, lut, kn, khat); break;
                case 3: prefill_decode_k<3, true>(raw, U, lane, pools, lut, kn, khat); break;
                case 4: prefill_decode_k<4, true>(raw, U, lane, pools, lut, kn, khat); break;
                case 5: prefill_decode_k<5, true>(raw, U, lane, pools, lut, kn, khat); break;
                case 6: prefill_decode_k<6, true>(raw, U, lane, pools, lut, kn, khat); break;
                case 7: prefill_decode_k<7, true>(raw, U, lane, pools, lut, kn, khat); break;
                default: prefill_decode_k<8, true>(raw, U, lane, pools, lut, kn, khat); break;
                }
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar[WS_KREADY]);
            mbar_wait(bar[WS_VFULL], par);
            if (t > 0) mbar_wait(bar[WS_ODONE], parp);               // PV(t-1) has consumed V^T
            {
                const __half *rv = reinterpret_cast<const __half *>(reinterpret_cast<const unsigned char *>(raw) + M.vnorm_off);
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    const int tau = 32 * q4 + lane;
                    vn[tau] = rv[(tau & 7) * 16 + (tau >> 4) * 2 + ((tau >> 3) & 1)];
                }
                __syncwarp();
                const uint32_t *vcodes = raw + (M.vcode_off >> 2);
                for (int v = pw; v < 16; v += kWsProducers) {
                    switch (b_v) {
                    case 1: prefill_decode_v<1, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    case 2: prefill_decode_v<2, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    case 3: prefill_decode_v<3, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    case 4: prefill_decode_v<4, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    case 5: prefill_decode_v<5, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    case 6: prefill_decode_v<6, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    case 7: prefill_decode_v<7, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    default: prefill_decode_v<8, true>(vcodes, v >> 1, lane, pools, lut, vn, vhat_t, v & 1); break;
                    }
                }
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar[WS_VREADY]);
        }
    } else {
        // ================= softmax: one thread per query row
        const int quad = warp & 3, rt = warp >> 2;
        const int row = 32 * quad + lane, crow = rt * 128 + row;
        const int64_t prow = pos0 + i_first + crow / G;             // position of this row's query token
        const uint32_t t_s = tm + ((uint32_t)(32 * quad) << 16) + (uint32_t)(rt * 128), t_o = t_s + RT * 128u;
        unsigned char *prow_s = ps + rt * 32768 + row * 128;
        float m_run = -INFINITY, l_run = 0.f;
        for (int t = 0; t < n_tiles; ++t) {
            const uint32_t par = t & 1, parp = (t - 1) & 1;
            mbar_wait(bar[WS_SFULL], par);
            tc_fence_after();
            const int rel = (int)max((int64_t)-1, min((int64_t)1 << 20, prow - (int64_t)t * kTile));   // columns > rel are in the future
            const bool nomask = __all_sync(0xFFFFFFFFu, rel >= 127);
            float alpha = 1.f, ls = 0.f;
            bool two_pass = t == 0 || !nomask, s_freed = false;
            if (!two_pass) {
                // ---- ONE pass over S with the running REFERENCE m_run instead of this tile's maximum: p = 2^(s - m_run).  softmax
                // does not care which reference is subtracted as long as nothing overflows; a row whose tile maximum exceeds the
                // reference by more than 2^8 (p would leave the comfortable fp16 range) sends the warp to the two-pass path below,
                // which moves the reference and rescales O.  Saves the second TMEM read and the max -> exp dependency; the next
                // chunk's tcgen05.ld is in flight while this chunk's exponentials run.
                float mx = -INFINITY;
                uint32_t sa[32], sb[32];
                tmem_ld32(t_s, sa);
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    uint32_t (&cur)[32] = (ch & 1) ? sb : sa;
                    uint32_t (&nxt)[32] = (ch & 1) ? sa : sb;
                    if (ch < 3) tmem_ld32(t_s + 32 * (ch + 1), nxt);
                    else {                                               // the last chunk is in registers: decide now, then S(t+1) may be issued
#pragma unroll
                        for (int i = 0; i < 32; i += 2) mx = fmax3(mx, __uint_as_float(cur[i]), __uint_as_float(cur[i + 1]));
                        two_pass = __any_sync(0xFFFFFFFFu, mx > m_run + 8.f);
                        if (two_pass) break;                             // (S is read again below: it must not be released)
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar[WS_SFREE]);
                        s_freed = true;
                    }
                    if (ch == 0) { mbar_wait(bar[WS_ODONE], parp); tc_fence_after(); }   // before the first P store: PV(t-1) has consumed P
#pragma unroll
                    for (int j = 0; j < 4; ++j) {                        // 8 tokens = one 16-byte chunk of the P row
                        float p[8];
#pragma unroll
                        for (int e = 0; e < 8; e += 2) {
                            const float x0 = __uint_as_float(cur[8 * j + e]), x1 = __uint_as_float(cur[8 * j + e + 1]);
                            if (ch < 3) mx = fmax3(mx, x0, x1);
                            p[e] = fast_exp2(x0 - m_run); p[e + 1] = fast_exp2(x1 - m_run);
                            ls += p[e] + p[e + 1];
                        }
                        const uint4 v = make_uint4(pack_half2(p[0], p[1]), pack_half2(p[2], p[3]), pack_half2(p[4], p[5]), pack_half2(p[6], p[7]));
                        const int col = 32 * ch + 8 * j;
                        *reinterpret_cast<uint4 *>(prow_s + (col >> 6) * 16384 + ((((col & 63) >> 3) ^ (row & 7)) << 4)) = v;
                    }
                }
            }
            if (two_pass) {
                float mx = -INFINITY;
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    uint32_t sr[32];
                    tmem_ld32(t_s + 32 * ch, sr);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (nomask) {
#pragma unroll
                        for (int i = 0; i < 32; i += 2) mx = fmax3(mx, __uint_as_float(sr[i]), __uint_as_float(sr[i + 1]));
                    } else {
#pragma unroll
                        for (int i = 0; i < 32; ++i) mx = fmaxf(mx, 32 * ch + i > rel ? -INFINITY : __uint_as_float(sr[i]));
                    }
                }
                const float mn = fmaxf(m_run, mx);                       // finite: tile 0 holds position 0
                alpha = fast_exp2(m_run - mn);
                m_run = mn;
                if (t > 0) { mbar_wait(bar[WS_ODONE], parp); tc_fence_after(); }    // PV(t-1) has consumed P; O is stable (a no-op after a one-pass attempt)
                ls = 0.f;
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    uint32_t sr[32];
                    tmem_ld32(t_s + 32 * ch, sr);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int j = 0; j < 4; ++j) {                        // 8 tokens = one 16-byte chunk of the P row
                        float p[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            const int i = 32 * ch + 8 * j + e;
                            p[e] = (!nomask && i > rel) ? 0.f : fast_exp2(__uint_as_float(sr[8 * j + e]) - mn);
                            ls += p[e];
                        }
                        const uint4 v = make_uint4(pack_half2(p[0], p[1]), pack_half2(p[2], p[3]), pack_half2(p[4], p[5]), pack_half2(p[6], p[7]));
                        const int col = 32 * ch + 8 * j;
                        *reinterpret_cast<uint4 *>(prow_s + (col >> 6) * 16384 + ((((col & 63) >> 3) ^ (row & 7)) << 4)) = v;
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0 && !s_freed) mbar_arrive(bar[WS_SFREE]);   // S(t+1) may be issued while O is rescaled
            l_run = fmaf(l_run, alpha, ls);
            if (t > 0 && __any_sync(0xFFFFFFFFu, alpha != 1.f)) {    // a row maximum moved: rescale O in place
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    uint32_t o[32];
                    tmem_ld32(t_o + 32 * ch, o);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                    tmem_st32(t_o + 32 * ch, o);
                }
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            }
            fence_proxy_async();                                     // P -> visible to the MMA
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar[WS_PREADY]);
        }
        // ---- normalise and store the rotated-domain output rows (fp32); derotate_kernel finishes them
        mbar_wait(bar[WS_ODONE], (n_tiles - 1) & 1);
        tc_fence_after();
        const float inv = 1.f / l_run;
        const int ti = i_first + crow / G, n = crow % G;
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
            uint32_t o[32];
            tmem_ld32(t_o + 32 * ch, o);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (ti < P.n_q) {
                float4 *dst = reinterpret_cast<float4 *>(P.opart + (((size_t)b * P.n_q + ti) * (P.Hkv * G) + h * G + n) * kDh + 32 * ch);
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    dst[i] = make_float4(__uint_as_float(o[4 * i]) * inv, __uint_as_float(o[4 * i + 1]) * inv,
                                         __uint_as_float(o[4 * i + 2]) * inv, __uint_as_float(o[4 * i + 3]) * inv);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tm) : "memory");
}

// out[row][k] = sum_j Pi^(128)[j][k] * o'[row][j] / sqrt(128)  ->  bf16  (the V de-rotation, once per output row)
__global__ void __launch_bounds__(128)
derotate_kernel(const float *__restrict__ opart, const float *__restrict__ rot128, int64_t n_rows,
                __nv_bfloat16 *__restrict__ out)
{
    __shared__ float o[4][kDh];
    const int d = threadIdx.x;
    const int64_t row0 = (int64_t)blockIdx.x * 4;
#pragma unroll
    for (int r = 0; r < 4; ++r) o[r][d] = row0 + r < n_rows ? opart[(row0 + r) * kDh + d] : 0.f;
    __syncthreads();
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 16
    for (int j = 0; j < kDh; ++j) {
        const float p = __ldg(rot128 + j * kDh + d);
#pragma unroll
        for (int r = 0; r < 4; ++r) acc[r] = fmaf(p, o[r][j], acc[r]);
    }
#pragma unroll
    for (int r = 0; r < 4; ++r)
        if (row0 + r < n_rows) out[(row0 + r) * kDh + d] = __float2bfloat16(acc[r] * 0.08838834764831845f);
}

size_t prefill_ws_bytes(const bgtq_layout *lay, int batch, int n_q)
{
    const size_t rows = (size_t)batch * n_q;
    return rows * lay->n_kv_heads * 8 * kDh * sizeof(__half) + rows * lay->n_q_heads * kDh * sizeof(float);
}

int launch_prefill(const bgtq_layout *lay, int layer, const void *cache, const void *q, const int32_t *seq_len,
                   int batch, int n_q, int64_t max_tokens, float scale, void *out, void *ws, size_t ws_bytes,
                   cudaStream_t st)
{
    const int Hkv = lay->n_kv_heads, Hq = lay->n_q_heads, G = Hq / Hkv;
    if (G != 1 && G != 2 && G != 4 && G != 8) { set_error("bgtq_prefill_attention: GQA group must be 1, 2, 4 or 8"); return BGTQ_EINVAL; }
    if (ws_bytes < prefill_ws_bytes(lay, batch, n_q)) { set_error("bgtq_prefill_attention: workspace too small"); return BGTQ_EWORKSPACE; }
    if (batch > 65535 || (int64_t)batch * n_q * Hkv > 0x7FFFFFFF / 8) { set_error("bgtq_prefill_attention: too many rows"); return BGTQ_EINVAL; }
    const size_t rows = (size_t)batch * n_q;
    __half *qp = reinterpret_cast<__half *>(ws);
    float *opart = reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(ws) + rows * Hkv * 8 * kDh * sizeof(__half));
    const HeadMeta *metas = lay->d_meta + (size_t)layer * Hkv;
    // q' for every query token: the decode q-fold with (batch * n_q) rows, plain layout
    qfold_kernel<1><<<(unsigned)(rows * Hkv * G), kDh, 0, st>>>(metas, lay->d_rot_t, (const __nv_bfloat16 *)q, (int)rows, Hkv, Hq,
                                                             scale * 1.4426950408889634f, qp, 1);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    const int raw_bytes = (lay->max_stride + 127) / 128 * 128;
    // two 128-row query tiles per CTA (warp-specialised kernel) when the raw tile still fits beside 192 KB of operands
    // (12.5 KB of static tables) and there is more than one tile of query rows; else one tile per CTA
    const int RT = (tc_operand_bytes(2) + raw_bytes + 13 * 1024 <= 227 * 1024 && (n_q * G > 128)) ? 2 : 1;
    const size_t smem = (size_t)tc_operand_bytes(RT) + (size_t)raw_bytes;
    if (first_use_on_device(3)) {
        CUDA_TRY(cudaFuncSetAttribute(prefill_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc_operand_bytes(1) + 40 * 1024));
        CUDA_TRY(cudaFuncSetAttribute(prefill_ws_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 13 * 1024));
    }
    PrefillParams P;
    P.metas = metas; P.cache = (const uint8_t *)cache; P.qp = qp; P.seq_len = seq_len; P.cb16 = lay->d_cb16;
    P.opart = opart; P.n_cap = (max_tokens + kTile - 1) / kTile; P.batch = batch; P.n_q = n_q; P.Hkv = Hkv; P.G = G;
    P.raw_bytes = raw_bytes;
    const int TQ = RT * 128 / G;
    dim3 grid((n_q + TQ - 1) / TQ, Hkv, batch);
    // a sequence shorter than the chunk (seq_len < n_q, a caller error the host cannot see) leaves its rows untouched
    // in the kernels: start from zeros so that the output is defined
    CUDA_TRY(cudaMemsetAsync(opart, 0, rows * Hq * kDh * sizeof(float), st));
    if (RT == 2) prefill_ws_kernel<<<grid, kWsThreads, smem, st>>>(P);
    else prefill_tc_kernel<1><<<grid, kTcThreads, smem, st>>>(P);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    derotate_kernel<<<(unsigned)((rows * Hq + 3) / 4), 128, 0, st>>>(opart, lay->d_rot + rot_offset(kDh), (int64_t)(rows * Hq),
                                                                      (__nv_bfloat16 *)out);
    count_launch();
    CUDA_TRY(cudaGetLastError());
    return BGTQ_OK;
}

// ---------------------------------------------------------------- test hook: the kernel's unpack routine
template <int B>
__device__ void debug_decode_b(const uint32_t *words, const uint32_t *pools, const uint16_t *lut, float *values)
{
    const int lane = threadIdx.x;
    uint32_t w[B], h[16];
    for (int i = 0; i < B; ++i) w[i] = words[i * 32 + lane];
    decode_unit<B>(w, pools, lut, h);
    for (int j = 0; j < 16; ++j) {
        const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&h[j]));
        values[lane * 32 + 2 * j] = f.x;
        values[lane * 32 + 2 * j + 1] = f.y;
    }
}
__global__ void debug_decode_kernel(int b, const uint32_t *words, const uint16_t *cb16, float *values)
{
    __shared__ __align__(16) uint16_t lut[kLutHalves];
    __shared__ uint32_t pools[16];
    build_lut(cb16, lut, threadIdx.x, 32);
    __syncwarp();
    if (threadIdx.x == 0) build_pools(lut, pools);
    __syncwarp();
    switch (b) {
    case 1: debug_decode_b<1>(words, pools, lut, values); break;
    case 2: debug_decode_b<2>(words, pools, lut, values); break;
    case 3: debug_decode_b<3>(words, pools, lut, values); break;
    case 4: debug_decode_b<4>(words, pools, lut, values); break;
    case 5: debug_decode_b<5>(words, pools, lut, values); break;
    case 6: debug_decode_b<6>(words, pools, lut, values); break;
    case 7: debug_decode_b<7>(words, pools, lut, values); break;
    default: debug_decode_b<8>(words, pools, lut, values); break;
    }
}

int debug_decode_unit(int b, const uint32_t *words, float *values)
{
    uint32_t *dw = nullptr; float *dv = nullptr; uint16_t *dcb = nullptr;
    std::vector<uint16_t> cb16(512, 0);
    for (int bb = 0; bb <= BGTQ_MAX_WIDTH; ++bb) {
        double lv[256];
        codebook_levels(bb, lv);
        for (int k = 0; k < (1 << bb); ++k) cb16[(1 << bb) - 1 + k] = __half_as_ushort(__double2half(lv[k]));
    }
    cudaError_t e = cudaMalloc(&dw, b * 32 * 4);
    if (e == cudaSuccess) e = cudaMalloc(&dv, 32 * 32 * 4);
    if (e == cudaSuccess) e = cudaMalloc(&dcb, 512 * 2);
    if (e == cudaSuccess) e = cudaMemcpy(dw, words, b * 32 * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dcb, cb16.data(), 512 * 2, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) { debug_decode_kernel<<<1, 32>>>(b, dw, dcb, dv); count_launch(); e = cudaGetLastError(); }
    if (e == cudaSuccess) e = cudaMemcpy(values, dv, 32 * 32 * 4, cudaMemcpyDeviceToHost);
    cudaFree(dw); cudaFree(dv); cudaFree(dcb);
    if (e != cudaSuccess) return cuda_fail(e, "bgtq_debug_decode_unit");
    return BGTQ_OK;
}

}  // namespace bgtq
