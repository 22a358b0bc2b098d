// bgtq_append.cu -- quantize-on-append: TQ-MSE per same-width K group and for V
// (PAPER.md:49, 108), packed into the BGTQ-v1 or BGTQ-v2 tile layout (DESIGN.md sections 4, 4b).
//
// Exactness: the arithmetic is the fp64 sequence of DESIGN.md section 3 -- fma chains in index
// order, IEEE sqrt / divide, strict '>' against tau_k * sigma -- written with explicit
// round-to-nearest intrinsics so the compiler cannot contract or reorder it.
//
// One CTA owns one (sequence, KV head, 128-token tile): it stages the tile in shared memory
// (loading the older tokens if the tile is partly filled), processes the new tokens in sub-batches
// of 16 (one m-tile of the decode kernel's fragment order), and writes the tile back with
// coalesced 16-byte stores.  No global atomics; every rotation row is read once per 16 tokens.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "bgtq_internal.h"

namespace bgtq {

#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

#ifndef BGTQ_APPEND_PHASES
#define BGTQ_APPEND_PHASES 0
#endif
constexpr int kAppendThreads = 256;
constexpr int kMetaBytes = (int)((sizeof(HeadMeta) + 15) / 16 * 16);
static_assert(sizeof(HeadMeta) % 4 == 0, "HeadMeta is copied word by word");
constexpr int kSub = 16;                       // tokens per sub-batch
constexpr int kMaxUnits = 2 * kMaxKSteps;

struct UnitDesc { uint16_t off; uint8_t b, nc; uint16_t ustart, pad; };   // ustart: grouped-order coordinate of slot q=0,c=0 (8 bytes: shared memory is what caps this kernel at 4 CTAs per SM)

// position of bit `bit` of the field of slot k in a unit of width b (DESIGN.md section 4 table)
__device__ __forceinline__ void field_bit_pos(int b, int k, int bit, int &word, int &pos)
{
    if (b == 1) { word = 0; pos = (15 - (k >> 1)) + 16 * (k & 1); }
    else if (b == 2) {
        int kk = k & 15, Q = kk >> 2, e = kk & 3;
        word = k >> 4; pos = 4 * ((Q & 1) * 4 + e) + 2 * (Q >> 1) + bit;
    } else if (b == 3 || (b == 4 && bit < 3)) {
        if (k < 24) { word = k >> 3; pos = 4 * (k & 7) + bit; }
        else { word = bit; pos = 4 * (k - 24) + 3; }
    } else if (b == 4) { word = 3; pos = 8 * (k & 3) + 7 - (k >> 2); }
    else { int s = b * k + bit; word = s >> 5; pos = s & 31; }
}

// write code idx into slot k of the unit whose word w lives at base[w * wstride] (32-bit words)
__device__ __forceinline__ void put_field(uint32_t *base, int wstride, int b, int k, unsigned idx)
{
    unsigned f = idx;
    if (b == 4) f = idx >= 8 ? (idx - 8) : (8u | (7u - idx));       // sign-magnitude storage
    for (int bit = 0; bit < b; ++bit) {
        int word, pos;
        field_bit_pos(b, k, bit, word, pos);
        uint32_t v = base[word * wstride];
        v = (v & ~(1u << pos)) | (((f >> bit) & 1u) << pos);
        base[word * wstride] = v;
    }
}

// The four slots 4i .. 4i+3 of a unit (one sub-batch's contribution to a lane: two tokens x two coordinates for K, four
// tokens for V) written with one read-modify-write per word they touch instead of one per bit: at every width the four
// fields are neighbours (DESIGN.md section 4 table).  pm: which of the four are present (tokens of this call).
__device__ __forceinline__ void rmw(uint32_t *w, uint32_t val, uint32_t mask) { if (mask) *w = (*w & ~mask) | val; }
__device__ __forceinline__ void pack4(uint32_t *wb, int ws, int b, int i, const unsigned (&f)[4], unsigned pm)
{
    uint32_t val = 0, mask = 0;
    if (b == 1) {                                                  // slot 2j+e at bit (15-j) + 16e
#pragma unroll
        for (int s = 0; s < 4; ++s)
            if ((pm >> s) & 1) { const int pos = 15 - (2 * i + (s >> 1)) + 16 * (s & 1); val |= (f[s] & 1u) << pos; mask |= 1u << pos; }
        rmw(wb, val, mask);
    } else if (b == 2) {                                           // word i>>2; Q = i&3, e = s
#pragma unroll
        for (int s = 0; s < 4; ++s)
            if ((pm >> s) & 1) { const int pos = 4 * ((i & 1) * 4 + s) + 2 * ((i & 3) >> 1); val |= (f[s] & 3u) << pos; mask |= 3u << pos; }
        rmw(wb + (i >> 2) * ws, val, mask);
    } else if (b <= 4) {
        unsigned g[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) g[s] = b == 4 ? (f[s] >= 8 ? f[s] - 8 : (8u | (7u - f[s]))) : f[s];   // width 4: sign-magnitude
        if (i < 6) {                                               // slots 0..23: word k>>3, nibble k&7
#pragma unroll
            for (int s = 0; s < 4; ++s)
                if ((pm >> s) & 1) { const int pos = 4 * ((i & 1) * 4 + s); val |= (g[s] & 7u) << pos; mask |= 7u << pos; }
            rmw(wb + (i >> 1) * ws, val, mask);
        } else {                                                   // slots 24..31: bit j of the field at word j, bit 4(k-24)+3
#pragma unroll
            for (int bit = 0; bit < 3; ++bit) {
                val = 0; mask = 0;
#pragma unroll
                for (int s = 0; s < 4; ++s)
                    if ((pm >> s) & 1) { const int pos = 4 * (4 * (i - 6) + s) + 3; val |= ((g[s] >> bit) & 1u) << pos; mask |= 1u << pos; }
                rmw(wb + bit * ws, val, mask);
            }
        }
        if (b == 4) {                                              // sign of slot 4Q+e (Q = i, e = s): word 3, bit 8e+7-Q
            val = 0; mask = 0;
#pragma unroll
            for (int s = 0; s < 4; ++s)
                if ((pm >> s) & 1) { const int pos = 8 * s + 7 - i; val |= ((g[s] >> 3) & 1u) << pos; mask |= 1u << pos; }
            rmw(wb + 3 * ws, val, mask);
        }
    } else {                                                       // widths 5..8: bits [b*k, b*k+b) of the stream, k = 4i .. 4i+3
        unsigned long long v64 = 0, m64 = 0;
        const unsigned long long fm = (1ull << b) - 1ull;
#pragma unroll
        for (int s = 0; s < 4; ++s)
            if ((pm >> s) & 1) { v64 |= (unsigned long long)(f[s] & fm) << (s * b); m64 |= fm << (s * b); }
        const int start = 4 * i * b, word = start >> 5, sh = start & 31;
        rmw(wb + word * ws, (uint32_t)(v64 << sh), (uint32_t)(m64 << sh));
        if (sh + 4 * b > 32) rmw(wb + (word + 1) * ws, (uint32_t)(v64 >> (32 - sh)), (uint32_t)(m64 >> (32 - sh)));
    }
}

// BGTQ-v2: bits that code f at slot k of a chunk (width b, r slots) contributes to word j of the chunk
__device__ __forceinline__ void slot_bits_v2(int b, int r, int k, int j, unsigned f, uint32_t &val, uint32_t &mask)
{
    if (b == 1) {
        if (j == 0) { const int pos = 8 * (k & 3) + 7 - (k >> 2); val |= (f & 1u) << pos; mask |= 1u << pos; }
    } else if (b == 2) {
        if ((k >> 4) == j) {
            const int kk = k & 15, Q = kk >> 2, e = kk & 3, pos = 4 * ((Q & 1) * 4 + e) + 2 * (Q >> 1);
            val |= (f & 3u) << pos; mask |= 3u << pos;
        }
    } else if (b == 3 || b == 4) {
        if (b == 4) f = f >= 8 ? (f - 8) : (8u | (7u - f));            // sign-magnitude storage
        const int nwm = r > 24 ? 3 : (r + 7) / 8;
        if (j < nwm) {
            if (k < 24) {
                if ((k >> 3) == j) { const int pos = 4 * (k & 7); val |= (f & 7u) << pos; mask |= 7u << pos; }
            } else { const int pos = 4 * (k - 24) + 3; val |= ((f >> j) & 1u) << pos; mask |= 1u << pos; }
        } else if (b == 4) { const int pos = 8 * (k & 3) + 7 - (k >> 2); val |= ((f >> 3) & 1u) << pos; mask |= 1u << pos; }
    } else {
        const int sh = b * k - 32 * j;                                  // field = bits [b*k, b*k+b) of the stream
        const uint32_t fm = (1u << b) - 1u;
        if (sh >= 0 && sh < 32) { val |= f << sh; mask |= fm << sh; }
        else if (sh < 0 && sh > -b) { val |= f >> (-sh); mask |= fm >> (-sh); }
    }
}

// ---- fast path (FAST = true; bulk appends): z ~ X Pi^T of a 16-token sub-batch on the tensor cores, exact recheck near thresholds
// One work item = 16 outputs (two n-tiles sharing their A fragments) of one rotation group; mma.sync.m16n8k8 TF32 with hi/lo
// splits of both operands (the split of Pi is precomputed: rot_hl = {tf32(Pi), Pi - tf32(Pi)}, row-major like the rotation table).
struct FastItem { uint16_t x0; uint8_t m, n0, b, sidx, isv, pad; };   // x0: first column of the group in a row of xs; n0: first output
constexpr int kMaxFastItems = 32;              // sum_g ceil(m_g / 16) <= 16 for K, 8 for V
constexpr int kFastWarps = kAppendThreads / 32;
constexpr int kFastPerWarp = kMaxFastItems / kFastWarps;
constexpr int kFastQueue = kSub * 256;         // every (token, column) of a sub-batch may need the exact chain
// Three TF32 products per k-step (hi/lo splits of x and Pi; lo x lo dropped): |z - z_exact| <= ~1.3e-5 sqrt(m) sigma (dropped term
// 2^-22, TF32 truncation of the lo operands 2^-21, fp32 accumulation of 48 MMAs at <= 2^-22 of ||x|| each; ||x|| = sqrt(m) sigma
// bounds every partial sum); the guard band is 4.5x that plus the fp32 rounding of tau * sigma.  A code whose z is inside the
// band of a neighbouring threshold (0.1-2 % of the codes) is recomputed with the exact fp64 chain, so the packed bytes are
// identical to the exact kernel's.  (A single TF32 product with its 1.2e-3 sqrt(m) sigma worst-case band was measured too:
// 2-10 % rechecks, slower overall.)
__device__ __forceinline__ float fast_guard(int m) { return 6.0e-5f * sqrtf((float)m) + 2.0e-5f; }
__device__ __forceinline__ uint32_t tf32_rna(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__device__ __forceinline__ double to_f64(float v) { return (double)v; }
__device__ __forceinline__ double to_f64(__nv_bfloat16 v) { return (double)__bfloat162float(v); }

template <typename T, bool ROPE, bool PAGED, bool FAST>
__global__ void __launch_bounds__(kAppendThreads, FAST ? 3 : 4)
quantize_append_kernel(const HeadMeta *__restrict__ metas, uint8_t *__restrict__ cache,
                       const T *__restrict__ k_new, const T *__restrict__ v_new,
                       const double *__restrict__ cb64, const float *__restrict__ rot_t, int batch,
                       int n_new, int Hkv, const int32_t *__restrict__ seq_len, int64_t n_cap,
                       int64_t max_tokens, const int32_t *__restrict__ pages, int pstride, int64_t n_pages,
                       const float *__restrict__ rope_cos, const float *__restrict__ rope_sin, int pairing, int cb_exact,
                       int max_rows, const float2 *__restrict__ rot_hl, int skip_full)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x;
#if BGTQ_APPEND_PHASES
    long long aph_t[8] = {0, 0, 0, 0, 0, 0, 0, 0}, aph_last = clock64();
    int aph_cur = 7;
#define APH(i) do { const long long now_ = clock64(); aph_t[aph_cur] += now_ - aph_last; aph_last = now_; aph_cur = (i); } while (0)
#else
#define APH(i) do { } while (0)
#endif
    const int h = blockIdx.y % Hkv, lrel = blockIdx.y / Hkv, s = blockIdx.z;
    const int64_t t0 = seq_len[s];
    const int64_t t_end = min(t0 + (int64_t)n_new, max_tokens);
    const int64_t tile = t0 / kTile + blockIdx.x;
    const int64_t tile_lo = tile * kTile;
    const int64_t lo = max(t0, tile_lo), hi = min(t_end, tile_lo + kTile);
    if (lo >= hi) return;
    if (skip_full && lo == tile_lo && hi == tile_lo + kTile) return;      // whole tiles of new tokens: quantize_tile_kernel

    // shared memory carve-up
    double *xs = reinterpret_cast<double *>(smem);                       // [16][256]
    double *tau = xs + kSub * 256;                                       // [512] thresholds (C_b at 2^b-1)
    double *sigma = tau + 512;                                           // [16][ns], ns = K groups + V groups of this head (<= max_rows)
    uint16_t *nrm = reinterpret_cast<uint16_t *>(sigma + kSub * max_rows);   // [16][ns] (+pad)
    uint8_t *idxs = reinterpret_cast<uint8_t *>(nrm + kSub * max_rows + 8);  // [16][256]
    UnitDesc *units = reinterpret_cast<UnitDesc *>(idxs + kSub * 256);   // [32]
    int *n_units_p = reinterpret_cast<int *>(units + kMaxUnits);
    HeadMeta *Msp = reinterpret_cast<HeadMeta *>(n_units_p + 4);         // this head's static metadata (kMetaBytes)
    // exact-density codebooks: V has its own flat table (C_{w, m} of the V group of width w; 512 more thresholds); else V
    // shares the flat table of K
    double *tauV_own = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(Msp) + kMetaBytes);
    unsigned char *after_tabs = reinterpret_cast<unsigned char *>(Msp) + kMetaBytes + (cb_exact ? 512 * 8 : 0);
    // fast path: fp32 thresholds (K table, V table), work items, recheck queue
    float *tau32 = reinterpret_cast<float *>(after_tabs);                           // [2][512]
    FastItem *items = reinterpret_cast<FastItem *>(tau32 + 1024);                   // [kMaxFastItems]
    uint16_t *queue = reinterpret_cast<uint16_t *>(items + kMaxFastItems);          // [kFastQueue]
    int *qcount = reinterpret_cast<int *>(queue + kFastQueue);                      // [0] entries, [1] items
    uint32_t *tbuf = reinterpret_cast<uint32_t *>(after_tabs + (FAST ? 1024 * 4 + kMaxFastItems * sizeof(FastItem) + kFastQueue * 2 + 16 : 0));   // tile, `stride` bytes
    // The metadata is read many times by single threads (unit list, group search, radii); one coalesced copy into
    // shared memory replaces those dependent global-memory round trips -- they dominated the one-token append.
    {
        const uint32_t *msrc = reinterpret_cast<const uint32_t *>(metas + blockIdx.y);
        uint32_t *mdst = reinterpret_cast<uint32_t *>(Msp);
        for (int i = tid; i < (int)(sizeof(HeadMeta) / 4); i += kAppendThreads) mdst[i] = __ldg(msrc + i);
    }
    __syncthreads();
    const HeadMeta &M = *Msp;
    const int stride = M.tile_stride, ng = M.n_groups, kdim = M.kdim, b_v = M.b_v;     // (b_v: BGTQ-v2 packing only)
    const int nvg = M.n_vgroups, ns = ng + nvg;

    uint8_t *gtile = PAGED ? cache + n_pages * ((int64_t)M.layer_prefix + M.head_prefix) + (int64_t)pages[(int64_t)s * pstride + tile] * stride
                           : cache + n_cap * ((int64_t)batch * M.layer_prefix + (int64_t)s * M.layer_sum + M.head_prefix) + tile * stride;
    {   // stage the tile: older tokens present -> load, else start from zeros
        const bool has_old = tile_lo < t0;
        const uint4 *src = reinterpret_cast<const uint4 *>(gtile);
        uint4 *dst = reinterpret_cast<uint4 *>(tbuf);
        for (int i = tid; i < stride / 16; i += kAppendThreads)
            dst[i] = has_old ? src[i] : make_uint4(0, 0, 0, 0);
    }
    // thresholds tau_k = (C[k] + C[k+1]) / 2 (exact in fp64); stored at the level's flat index
    const double *cbK = cb64 + (cb_exact ? (size_t)blockIdx.y * 1024 : 0);     // this head's tables (exact: [K 512 | V 512])
    for (int i = tid; i < 511; i += kAppendThreads) {
        double c0 = cbK[i], c1 = cbK[i + 1 < 511 ? i + 1 : i];
        tau[i] = __dmul_rn(__dadd_rn(c0, c1), 0.5);
    }
    if (cb_exact) {
        const double *cbV = cbK + 512;
        for (int i = tid; i < 511; i += kAppendThreads) tauV_own[i] = __dmul_rn(__dadd_rn(cbV[i], cbV[i + 1 < 511 ? i + 1 : i]), 0.5);
    }
    const double *tauV = cb_exact ? tauV_own : tau;
    if (tid == 0) {  // list of half-step units of the K code section
        int n = 0, j = 0;
        for (int ks = 0; ks < (M.format == 2 ? 0 : M.n_ksteps); ++ks) {   // (BGTQ-v2 packs from M.chunks, step 5)
            const KStep &K = M.ksteps[ks];
            int g = K.flags >> 4;
            if (K.flags & 1) j = 0;
            units[n++] = UnitDesc{K.off0, K.b, K.nc0, (uint16_t)(M.gstart[g] + 8 * j), 0};
            ++j;
            if (K.off1 != 0xFFFF) { units[n++] = UnitDesc{K.off1, K.b, K.nc1, (uint16_t)(M.gstart[g] + 8 * j), 0}; ++j; }
        }
        *n_units_p = n;
        if (FAST) {                               // n-tiles of every rotation group of this head
            int ni = 0;
            for (int g = 0; g < ng; ++g)
                for (int n0 = 0; n0 < M.gm[g]; n0 += 16) items[ni++] = FastItem{M.gstart[g], (uint8_t)M.gm[g], (uint8_t)n0, M.gb[g], (uint8_t)g, 0, 0};
            for (int gv = 0; gv < nvg; ++gv)
                for (int n0 = 0; n0 < 16 * M.vgcnt[gv]; n0 += 16)
                    items[ni++] = FastItem{(uint16_t)(128 + 16 * M.vgstart[gv]), (uint8_t)(16 * M.vgcnt[gv]), (uint8_t)n0, M.vgb[gv], (uint8_t)(ng + gv), 1, 0};
            qcount[1] = ni;
        }
    }
    __syncthreads();
    if (FAST)
        for (int i = tid; i < 1022; i += kAppendThreads) tau32[i + (i >= 511 ? 1 : 0)] = (float)(i < 511 ? tau[i] : tauV[i - 511]);
    const int n_items = FAST ? qcount[1] : 0;
    const int n_units = *n_units_p;

    // this thread's row of the rotation: col < kdim -> K group row, col >= 128 -> row of its V group (grouped V order)
    const int col = tid;
    int my_m = 0, my_r = 0, my_x0 = 0, my_g = 0, my_b = 0;
    if (col >= 128) {
        const int gv = M.vbg[(col - 128) >> 4];
        my_m = 16 * M.vgcnt[gv]; my_x0 = 128 + 16 * M.vgstart[gv]; my_r = col - my_x0; my_g = ng + gv; my_b = M.vgb[gv];
    }
    else if (col < kdim) {
        int g = 0;
        while (g + 1 < ng && col >= M.gstart[g + 1]) ++g;
        my_m = M.gm[g]; my_r = col - M.gstart[g]; my_x0 = M.gstart[g]; my_g = g; my_b = M.gb[g];
    }
    const float *myrot = rot_t + rot_offset(my_m > 0 ? my_m : 2) + my_r;
    // gather source of column `col`: V coordinate col-128, or the K coordinate stored at grouped position col
    const T *g_src = col >= 128 ? v_new : k_new;
    const int g_off = col >= 128 ? 16 * M.vblk[(col - 128) >> 4] + (col & 15) : (col < kdim ? (int)M.coords[col] : -1);
    int g_part = -1, g_blk = 0;
    bool g_isb = false;
    if (ROPE && col < kdim) {               // RoPE partner of this K coordinate, its block and which member it is
        const bool half = pairing == BGTQ_PAIR_HALF;
        g_blk = half ? (g_off & (kDh / 2 - 1)) : (g_off >> 1);
        g_isb = half ? (g_off >= kDh / 2) : (g_off & 1);
        g_part = half ? (g_off ^ (kDh / 2)) : (g_off ^ 1);
    }

    for (int i = 0; i < kTile / kSub; ++i) {
        const int64_t base = tile_lo + i * kSub;
        const int64_t nlo = max(lo, base), nhi = min(hi, base + kSub);
        if (nlo >= nhi) continue;
        APH(0);
        // ---- 1. gather the sub-batch: xs[tt][0..127] = K in grouped order, xs[tt][128..255] = V.  Thread c owns
        //      (grouped V order) column c (its source coordinate is fixed), so the kSub loads are independent and in flight together.
        {
            const int64_t row0 = ((((int64_t)lrel * batch + s) * n_new + (base - t0)) * Hkv + h) * kDh;
            const int64_t rstep = (int64_t)Hkv * kDh;
#pragma unroll 4
            for (int tt = 0; tt < kSub; ++tt) {
                const int64_t tok = base + tt;
                double v = 0.0;
                if (tok >= nlo && tok < nhi && g_off >= 0) {
                    const int64_t row = row0 + tt * rstep;
                    v = to_f64(g_src[row + g_off]);
                    if constexpr (ROPE) {
                        // fused RoPE: block i = pair (a, b); a' = x_a cos - x_b sin, b' = x_a sin + x_b cos
                        // at position tok.  Inputs and table entries have <= 24-bit significands, so both products
                        // are exact in fp64 and each output is the correctly rounded value of the exact expression.
                        if (g_part >= 0) {
                            const double xp = to_f64(k_new[row + g_part]);
                            const double cs = (double)__ldg(rope_cos + tok * (kDh / 2) + g_blk);
                            const double sn = (double)__ldg(rope_sin + tok * (kDh / 2) + g_blk);
                            v = g_isb ? __dadd_rn(__dmul_rn(xp, sn), __dmul_rn(v, cs)) : __dadd_rn(__dmul_rn(v, cs), -__dmul_rn(xp, sn));
                        }
                    }
                }
                xs[tt * 256 + tid] = v;
            }
        }
        __syncthreads();
        APH(1);
        // ---- 2. radii: ss = fma chain, r = sqrt(ss), sigma = r / sqrt(m), h = fp16_rne_sat(r)
        if (tid < kSub * ns && base + tid / ns >= nlo && base + tid / ns < nhi) {
            int tt = tid / ns, g = tid % ns;
            int x0 = g < ng ? M.gstart[g] : 128 + 16 * M.vgstart[g - ng], m = g < ng ? M.gm[g] : 16 * M.vgcnt[g - ng];
            const double *x = xs + tt * 256 + x0;
            double ss = 0.0;
            for (int j = 0; j < m; ++j) ss = __fma_rn(x[j], x[j], ss);
            double r = __dsqrt_rn(ss);
            sigma[tt * ns + g] = __ddiv_rn(r, __dsqrt_rn((double)m));
            __half hv = __double2half(r);
            uint16_t hb = __half_as_ushort(hv);
            if (r >= 65520.0) hb = 0x7BFF;
            nrm[tt * ns + g] = hb;
        }
        const int tt_lo = (int)(nlo - base), tt_hi = (int)(nhi - base);
        if constexpr (FAST) {
            APH(2);
            // ---- 3'. z ~ X Pi^T on the tensor cores: warp w takes items w, w+8, ...; accumulators stay in registers
            const int warp = tid >> 5, lane = tid & 31, fg = lane >> 2, fc = lane & 3;
            if (tid == 0) qcount[0] = 0;
            float acc[kFastPerWarp][2][4];
#pragma unroll
            for (int ii = 0; ii < kFastPerWarp; ++ii) {
#pragma unroll
                for (int e = 0; e < 4; ++e) acc[ii][0][e] = acc[ii][1][e] = 0.f;
                const int item = warp + ii * kFastWarps;
                if (item < n_items) {
                    const FastItem it = items[item];
                    const int m = it.m, nA = it.n0 + fg, nB = nA + 8;
                    const bool two = it.n0 + 8 < m;                                // (warp-uniform) the second n-tile exists
                    const double *xa = xs + fg * 256 + it.x0;                     // token row fg; row fg + 8 is 8 * 256 further
                    const float2 *RA = rot_hl + rot_offset(m) + (size_t)(nA < m ? nA : 0) * m;   // B(k, n) = Pi^(m)[n][k]
                    const float2 *RB = rot_hl + rot_offset(m) + (size_t)(nB < m ? nB : 0) * m;
                    // operand pointers of this lane: B rows are clamped to row 0 for outputs beyond the group (their accumulators
                    // are never read), so the full k-steps need no predicates at all; only a ragged last k-step is masked
                    const float2 *pA = RA + fc, *pB = RB + fc;
                    const double *px = xa + fc;
                    auto kstep = [&](const float2 ca0, const float2 ca1, const float2 cb0, const float2 cb1,
                                     const float a0, const float a1, const float a2, const float a3) {
                        const uint32_t ah[4] = {tf32_rna(a0), tf32_rna(a1), tf32_rna(a2), tf32_rna(a3)};
                        const uint32_t al[4] = {__float_as_uint(a0 - __uint_as_float(ah[0])), __float_as_uint(a1 - __uint_as_float(ah[1])),
                                                __float_as_uint(a2 - __uint_as_float(ah[2])), __float_as_uint(a3 - __uint_as_float(ah[3]))};
                        mma_tf32(acc[ii][0], al, __float_as_uint(ca0.x), __float_as_uint(ca1.x));   // small terms first
                        mma_tf32(acc[ii][0], ah, __float_as_uint(ca0.y), __float_as_uint(ca1.y));
                        mma_tf32(acc[ii][0], ah, __float_as_uint(ca0.x), __float_as_uint(ca1.x));
                        if (two) {
                            mma_tf32(acc[ii][1], al, __float_as_uint(cb0.x), __float_as_uint(cb1.x));
                            mma_tf32(acc[ii][1], ah, __float_as_uint(cb0.y), __float_as_uint(cb1.y));
                            mma_tf32(acc[ii][1], ah, __float_as_uint(cb0.x), __float_as_uint(cb1.x));
                        }
                    };
                    const int kfull = m & ~7;
#pragma unroll 2
                    for (int k0 = 0; k0 < kfull; k0 += 8)
                        kstep(__ldg(pA + k0), __ldg(pA + k0 + 4), __ldg(pB + k0), __ldg(pB + k0 + 4),
                              (float)px[k0], (float)px[8 * 256 + k0], (float)px[k0 + 4], (float)px[8 * 256 + k0 + 4]);
                    if (kfull < m) {                                   // ragged tail: k >= m contributes zero
                        const bool va = kfull + fc < m, vb = kfull + fc + 4 < m;
                        const float2 zero2 = make_float2(0.f, 0.f);
                        kstep(va ? __ldg(pA + kfull) : zero2, vb ? __ldg(pA + kfull + 4) : zero2,
                              va ? __ldg(pB + kfull) : zero2, vb ? __ldg(pB + kfull + 4) : zero2,
                              va ? (float)px[kfull] : 0.f, va ? (float)px[8 * 256 + kfull] : 0.f,
                              vb ? (float)px[kfull + 4] : 0.f, vb ? (float)px[8 * 256 + kfull + 4] : 0.f);
                    }
                }
            }
            __syncthreads();                                                       // sigma of step 2 is complete
            APH(3);
            // ---- 4'. codes from z where it is clear of the neighbouring thresholds; the rest go to the queue
#pragma unroll
            for (int ii = 0; ii < kFastPerWarp; ++ii) {
                const int item = warp + ii * kFastWarps;
                if (item < n_items) {
                    const FastItem it = items[item];
                    const float *tb = tau32 + (it.isv ? 512 : 0) + ((1 << it.b) - 1);
                    const float gc = fast_guard(it.m);
                    const int L = 1 << it.b;
                    // the eight searches of a lane side by side (the probes of one search are a dependent LDS -> FMUL -> FSETP chain)
                    float z8[8], sg8[8];
                    int a8[8];
                    bool ok[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const int tt = fg + 8 * ((e >> 1) & 1), nl = it.n0 + 8 * (e >> 2) + 2 * fc + (e & 1);
                        ok[e] = nl < it.m && tt >= tt_lo && tt < tt_hi;
                        z8[e] = acc[ii][e >> 2][e & 3];
                        sg8[e] = ok[e] ? (float)sigma[tt * ns + it.sidx] : 0.f;
                        a8[e] = 0;
                    }
                    for (int bit = it.b - 1; bit >= 0; --bit) {
                        const int step = 1 << bit;
#pragma unroll
                        for (int e = 0; e < 8; ++e)
                            if (z8[e] > tb[a8[e] + step - 1] * sg8[e]) a8[e] += step;
                    }
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        if (!ok[e]) continue;
                        const int tt = fg + 8 * ((e >> 1) & 1), col = it.x0 + it.n0 + 8 * (e >> 2) + 2 * fc + (e & 1);
                        const int a = a8[e];
                        const float z = z8[e], sg = sg8[e], gd = gc * sg;
                        const float tlo = tb[a > 0 ? a - 1 : 0] * sg, thi = tb[a < L - 1 ? a : 0] * sg;
                        const bool risky = (a > 0 && !(z - tlo > gd)) || (a < L - 1 && !(thi - z > gd));
                        idxs[tt * 256 + col] = (uint8_t)a;
                        if (risky) queue[atomicAdd(&qcount[0], 1)] = (uint16_t)((tt << 8) | col);
                    }
                }
            }
            __syncthreads();
            APH(4);
            // ---- 4''. the exact fp64 chain (oracle order) for the queued (token, column) pairs
            const int qn = qcount[0];
            for (int e = tid; e < qn; e += kAppendThreads) {
                const int ent = queue[e], tt = ent >> 8, col = ent & 255;
                int m, x0, sidx, b;
                const double *tb;
                if (col >= 128) {
                    const int gv = M.vbg[(col - 128) >> 4];
                    m = 16 * M.vgcnt[gv]; x0 = 128 + 16 * M.vgstart[gv]; sidx = ng + gv; b = M.vgb[gv]; tb = tauV + ((1 << b) - 1);
                } else {
                    int g = 0;
                    while (g + 1 < ng && col >= M.gstart[g + 1]) ++g;
                    m = M.gm[g]; x0 = M.gstart[g]; sidx = g; b = M.gb[g]; tb = tau + ((1 << b) - 1);
                }
                // row (col - x0) of Pi^(m), contiguous: hi + lo is the fp32 entry exactly; 16-byte loads, 16 in flight
                const float4 *Rq = reinterpret_cast<const float4 *>(rot_hl + rot_offset(m) + (size_t)(col - x0) * m);
                const double *x = xs + tt * 256 + x0;
                double zz = 0.0;
                int k = 0;
                for (; k + 32 <= m; k += 32) {
                    float4 pf[16];
#pragma unroll
                    for (int u = 0; u < 16; ++u) pf[u] = __ldg(Rq + (k >> 1) + u);
#pragma unroll
                    for (int u = 0; u < 16; ++u) {
                        zz = __fma_rn((double)(pf[u].x + pf[u].y), x[k + 2 * u], zz);
                        zz = __fma_rn((double)(pf[u].z + pf[u].w), x[k + 2 * u + 1], zz);
                    }
                }
                for (; k < m; k += 2) {                                          // (m is even)
                    const float4 p = __ldg(Rq + (k >> 1));
                    zz = __fma_rn((double)(p.x + p.y), x[k], zz);
                    zz = __fma_rn((double)(p.z + p.w), x[k + 1], zz);
                }
                const double sg = sigma[tt * ns + sidx];
                int a = 0;
                for (int bit = b - 1; bit >= 0; --bit)
                    if (zz > __dmul_rn(tb[a + (1 << bit) - 1], sg)) a += 1 << bit;
                idxs[tt * 256 + col] = (uint8_t)a;
            }
        } else {
            // ---- 3. rotation: z[tt] = fma chain over k of Pi[r][k] * x_k (k ascending: the oracle's order).
            //      Rotation rows are read 4 at a time ahead of the chain; a single new token (decode-time
            //      append) takes the scalar path so that the step is latency- not throughput-shaped.
            double z[kSub];
    #pragma unroll
            for (int tt = 0; tt < kSub; ++tt) z[tt] = 0.0;
            if (my_m > 0) {
                const double *x = xs + my_x0;
                if (tt_hi - tt_lo == 1) {
                    const double *x1 = x + tt_lo * 256;
                    double zz = 0.0;
                    int k = 0;
                    for (; k + 32 <= my_m; k += 32) {            // 32 independent loads in flight, then the chain
                        float pf[32];
    #pragma unroll
                        for (int u = 0; u < 32; ++u) pf[u] = __ldg(myrot + (size_t)(k + u) * my_m);
    #pragma unroll
                        for (int u = 0; u < 32; ++u) zz = __fma_rn((double)pf[u], x1[k + u], zz);
                    }
                    for (; k + 8 <= my_m; k += 8) {
                        float pf[8];
    #pragma unroll
                        for (int u = 0; u < 8; ++u) pf[u] = __ldg(myrot + (size_t)(k + u) * my_m);
    #pragma unroll
                        for (int u = 0; u < 8; ++u) zz = __fma_rn((double)pf[u], x1[k + u], zz);
                    }
                    for (; k < my_m; ++k) zz = __fma_rn((double)__ldg(myrot + (size_t)k * my_m), x1[k], zz);
    #pragma unroll
                    for (int tt = 0; tt < kSub; ++tt) if (tt == tt_lo) z[tt] = zz;
                } else {
                    int k = 0;
                    // blocks of 4 rotation entries, the next block's loads issued before this block's 64 chained FMAs:
                    // the table is an L2 hit (4 CTAs x 56 KB leave little L1), so its latency has to be covered
                    const int kend4 = my_m & ~3;
                    float pc[4];
                    if (kend4 > 0) {
    #pragma unroll
                        for (int u = 0; u < 4; ++u) pc[u] = __ldg(myrot + (size_t)u * my_m);
                    }
                    for (; k < kend4; k += 4) {
                        float pn[4];
                        const int kn = k + 4 < kend4 ? k + 4 : k;           // (the last block re-reads itself: no branch)
    #pragma unroll
                        for (int u = 0; u < 4; ++u) pn[u] = __ldg(myrot + (size_t)(kn + u) * my_m);
                        const double p0 = (double)pc[0], p1 = (double)pc[1], p2 = (double)pc[2], p3 = (double)pc[3];
    #pragma unroll
                        for (int tt = 0; tt < kSub; ++tt) {
                            const double2 xa = *reinterpret_cast<const double2 *>(x + tt * 256 + k);
                            const double2 xb = *reinterpret_cast<const double2 *>(x + tt * 256 + k + 2);
                            z[tt] = __fma_rn(p3, xb.y, __fma_rn(p2, xb.x, __fma_rn(p1, xa.y, __fma_rn(p0, xa.x, z[tt]))));
                        }
    #pragma unroll
                        for (int u = 0; u < 4; ++u) pc[u] = pn[u];
                    }
                    for (; k + 4 <= my_m; k += 4) {
                        float pf[4];
    #pragma unroll
                        for (int u = 0; u < 4; ++u) pf[u] = __ldg(myrot + (size_t)(k + u) * my_m);
                        const double p0 = (double)pf[0], p1 = (double)pf[1], p2 = (double)pf[2], p3 = (double)pf[3];
                        // x[tt][k..k+3] as two 16-byte loads (group starts are even and k is a multiple of 4, so the
                        // address is 16-byte aligned); per token the chain still runs over k in ascending order
    #pragma unroll
                        for (int tt = 0; tt < kSub; ++tt) {
                            const double2 xa = *reinterpret_cast<const double2 *>(x + tt * 256 + k);
                            const double2 xb = *reinterpret_cast<const double2 *>(x + tt * 256 + k + 2);
                            z[tt] = __fma_rn(p3, xb.y, __fma_rn(p2, xb.x, __fma_rn(p1, xa.y, __fma_rn(p0, xa.x, z[tt]))));
                        }
                    }
                    for (; k < my_m; ++k) {
                        const double pi = (double)__ldg(myrot + (size_t)k * my_m);
    #pragma unroll
                        for (int tt = 0; tt < kSub; ++tt) z[tt] = __fma_rn(pi, x[tt * 256 + k], z[tt]);
                    }
                }
            }
            __syncthreads();
            // ---- 4. scalar quantise: idx = #{k : z > tau_k * sigma}; the predicate is monotone in k
            if (my_m > 0) {
                const double *tb = (col >= 128 ? tauV : tau) + ((1 << my_b) - 1);
                // the count is found bit by bit (always my_b probes), all kSub searches side by side so that the
                // dependent LDS -> DMUL -> DSETP chains of different tokens overlap; same count as any other search
                // because the predicate is monotone in k
                const double *sgp = sigma + my_g;
                if (tt_hi - tt_lo == 1) {                         // decode-time append: one token, one search
                    double zz = 0.0;
    #pragma unroll
                    for (int tt = 0; tt < kSub; ++tt) if (tt == tt_lo) zz = z[tt];
                    const double sg = sgp[tt_lo * ns];
                    int a = 0;
                    for (int bit = my_b - 1; bit >= 0; --bit)
                        if (zz > __dmul_rn(tb[a + (1 << bit) - 1], sg)) a += 1 << bit;
                    idxs[tt_lo * 256 + col] = (uint8_t)a;
                } else
    #pragma unroll
                for (int t0h = 0; t0h < kSub; t0h += 8) {         // 8 searches side by side (register budget: 64)
                    int a[8];
    #pragma unroll
                    for (int tt = 0; tt < 8; ++tt) a[tt] = 0;
                    for (int bit = my_b - 1; bit >= 0; --bit) {
                        const int step = 1 << bit;
    #pragma unroll
                        for (int tt = 0; tt < 8; ++tt)
                            if (z[t0h + tt] > __dmul_rn(tb[a[tt] + step - 1], sgp[(t0h + tt) * ns])) a[tt] += step;
                    }
    #pragma unroll
                    for (int tt = 0; tt < 8; ++tt)
                        if (t0h + tt >= tt_lo && t0h + tt < tt_hi) idxs[(t0h + tt) * 256 + col] = (uint8_t)a[tt];
                }
            }
        }
        __syncthreads();
        APH(5);
        // ---- 5. pack the sub-batch's fields; each (unit, lane) word set has exactly one owner
        if (M.format == 2) {
            // BGTQ-v2: a K word belongs to one token (composed whole), a V word to one dimension and 32 tokens (read-modify-write)
            const int nch = M.n_ksteps, kq4 = M.kcode_bytes >> 4;        // words of one quadrant's K section
            for (int it = tid; it < kSub * nch * 8; it += kAppendThreads) {
                const int j = it & 7, ch = (it >> 3) % nch, tt = (it >> 3) / nch;
                const Chunk2 C2 = M.chunks[ch];
                const int64_t tok = base + tt;
                if (j >= C2.nw || tok < nlo || tok >= nhi) continue;
                const int tau = i * kSub + tt;
                uint32_t val = 0, mask = 0;
                const uint8_t *ip = idxs + tt * 256 + C2.ustart;
                for (int k = 0; k < C2.r; ++k) slot_bits_v2(C2.b, C2.r, k, j, ip[k], val, mask);
                tbuf[(tau >> 5) * kq4 + (C2.off >> 2) + j * 32 + (tau & 31)] = val;
            }
            const int c = i >> 1, k0 = (i & 1) * kSub;
            for (int it = tid; it < kDh * b_v; it += kAppendThreads) {
                const int d = it % kDh, j = it / kDh;
                uint32_t val = 0, mask = 0;
                for (int tt = tt_lo; tt < tt_hi; ++tt) slot_bits_v2(b_v, 32, k0 + tt, j, idxs[tt * 256 + 128 + d], val, mask);
                uint32_t *wp = tbuf + ((M.vcode_off + ((d >> 5) * 4 + c) * b_v * 128) >> 2) + j * 32 + (d & 31);
                *wp = (*wp & ~mask) | val;
            }
            if (tid < kSub * ns) {                                         // fp16 norms in natural token order (one V group)
                const int tt = tid / ns, g = tid % ns;
                const int64_t tok = base + tt;
                if (tok >= nlo && tok < nhi) {
                    const int off = g < ng ? M.knorm_off + 256 * g : M.vnorm_off;
                    reinterpret_cast<uint16_t *>(reinterpret_cast<uint8_t *>(tbuf) + off)[i * kSub + tt] = nrm[tt * ns + g];
                }
            }
            __syncthreads();
            continue;
        }
        const int kitems = n_units * 32;
        for (int it = tid; it < kitems + 16 * 32; it += kAppendThreads) {
            if (it < kitems) {
                const UnitDesc U = units[it >> 5];
                const int lp = it & 31, lanes = 8 * U.nc;
                if (lp >= lanes) continue;
                // lp = g8 * nc + c with nc in 1..4 lanes per row: no integer division (nc = 3: g8 = lp * 11 >> 5 for lp < 24)
                const int g8 = U.nc == 4 ? lp >> 2 : (U.nc == 2 ? lp >> 1 : (U.nc == 1 ? lp : (lp * 11) >> 5)), c = lp - g8 * U.nc;
                uint32_t *wbase = tbuf + (U.off >> 2) + lp;
                if constexpr (FAST) {
                    unsigned f[4], pm = 0;
#pragma unroll
                    for (int sl = 0; sl < 4; ++sl) {                   // slot 4i + 2p + q: token row 8p + g8, coordinate 2c + q
                        const int tt = 8 * (sl >> 1) + g8;
                        f[sl] = idxs[tt * 256 + U.ustart + 2 * c + (sl & 1)];
                        if (tt >= tt_lo && tt < tt_hi) pm |= 1u << sl;
                    }
                    pack4(wbase, lanes, U.b, i, f, pm);
                } else {                                               // (64-register budget: the word-wise packer makes the rotation loop spill)
                    for (int p = 0; p < 2; ++p) {
                        int tt = 8 * p + g8;
                        int64_t tok = base + tt;
                        if (tok < nlo || tok >= nhi) continue;
                        for (int q = 0; q < 2; ++q)
                            put_field(wbase, lanes, U.b, i * 4 + p * 2 + q, idxs[tt * 256 + U.ustart + 2 * c + q]);
                    }
                }
            } else {
                const int v = it - kitems, unit = v >> 5, lane = v & 31;   // unit = 2J' + rho, J' = grouped V block
                const int gq = lane >> 2, c = lane & 3;
                const int u = 16 * (unit >> 1) + 8 * (unit & 1) + gq;      // grouped V coordinate
                const int bw = M.vbw[unit >> 1];
                uint32_t *wbase = tbuf + ((M.vboff[unit >> 1] + (unit & 1) * 128 * bw) >> 2) + lane;
                if constexpr (FAST) {
                    unsigned f[4], pm = 0;
#pragma unroll
                    for (int sl = 0; sl < 4; ++sl) {                   // slot 4i + 2o + e: token row 8o + 2c + e
                        const int tt = 8 * (sl >> 1) + 2 * c + (sl & 1);
                        f[sl] = idxs[tt * 256 + 128 + u];
                        if (tt >= tt_lo && tt < tt_hi) pm |= 1u << sl;
                    }
                    pack4(wbase, 32, bw, i, f, pm);
                } else {
                    for (int o = 0; o < 2; ++o)
                        for (int e = 0; e < 2; ++e) {
                            int tt = 8 * o + 2 * c + e;
                            int64_t tok = base + tt;
                            if (tok < nlo || tok >= nhi) continue;
                            put_field(wbase, 32, bw, i * 4 + o * 2 + e, idxs[tt * 256 + 128 + u]);
                        }
                }
            }
        }
        if (tid < kSub * ns) {   // fp16 norms: token tau at entry (tau&7)*16 + (tau>>4)*2 + ((tau>>3)&1)
            int tt = tid / ns, g = tid % ns;
            int64_t tok = base + tt;
            if (tok >= nlo && tok < nhi) {
                int t128 = i * kSub + tt;
                int slot = (t128 & 7) * 16 + (t128 >> 4) * 2 + ((t128 >> 3) & 1);
                int off = g < ng ? M.knorm_off + 256 * g : M.vnorm_off + 256 * (g - ng);
                reinterpret_cast<uint16_t *>(reinterpret_cast<uint8_t *>(tbuf) + off)[slot] = nrm[tt * ns + g];
            }
        }
        __syncthreads();
    }
    APH(6);
    {   // write the tile back
        uint4 *dst = reinterpret_cast<uint4 *>(gtile);
        const uint4 *src = reinterpret_cast<const uint4 *>(tbuf);
        for (int i = tid; i < stride / 16; i += kAppendThreads) dst[i] = src[i];
    }
#if BGTQ_APPEND_PHASES
    APH(7);
    if ((tid == 0 || tid == 200) && blockIdx.x == 3 && blockIdx.y == 0 && blockIdx.z == 0)
        printf("append phases (tid %d, FAST %d): gather %lld radii %lld mma %lld quant %lld recheck %lld pack %lld writeback %lld setup %lld\n", tid, (int)FAST,
               aph_t[0], aph_t[1], aph_t[2], aph_t[3], aph_t[4], aph_t[5], aph_t[6], aph_t[7]);
#endif
#undef APH
}

// ---------------------------------------------------------------- bulk path: a whole tile per pass
// quantize_tile_kernel: one CTA (512 threads) quantises a tile whose 128 tokens are ALL new (bulk prefill appends), in ONE
// pass instead of eight 16-token sub-batches: every phase (gather, radii, rotation, threshold search, recheck, packing) runs
// once over 128 tokens, so its latency is paid once per tile and the rotation operands are read once per tile instead of
// eight times.  Same arithmetic as the FAST sub-batch path (three TF32 products with hi/lo splits, fast_guard band, exact
// fp64 chain in oracle order for every code inside the band; radii by the exact fp64 chains), hence the same bytes as the
// exact kernel.  Partly filled first / last tiles of the same call are left to quantize_append_kernel (skip_full = 1).
// Not for fused RoPE (the rotated keys are not fp32 values), paged caches or BGTQ-v2.
constexpr int kTileThreads = 512;
constexpr int kTileWarps = kTileThreads / 32;
constexpr int kXsLd = 260;                 // floats per token row of xs: 256 + 4, so the A-fragment reads (row g, column c) hit 32 banks
constexpr int kTileQueue = 6144;           // recheck queue; when more codes than that sit inside a band every code is rechecked
constexpr int kIdxLd = 260;                // bytes per token row of idxs: 256 + 4, so the packers' byte gathers (8 token rows per warp) hit 8 banks

// All B words of one lane of a unit from its 32 codes (slot k -> f[k]); the bit positions are DESIGN.md section 4's table
// (field_bit_pos), folded at compile time.
template <int B>
__device__ __forceinline__ void pack_unit(const unsigned (&f)[32], uint32_t (&w)[B])
{
#pragma unroll
    for (int j = 0; j < B; ++j) w[j] = 0u;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        const unsigned g = B == 4 ? (f[k] >= 8 ? f[k] - 8 : (8u | (7u - f[k]))) : f[k];   // width 4: sign-magnitude storage
#pragma unroll
        for (int bit = 0; bit < B; ++bit) {
            int word, pos;
            field_bit_pos(B, k, bit, word, pos);
            w[word] |= ((g >> bit) & 1u) << pos;
        }
    }
}
template <int B>
__device__ __forceinline__ void pack_store(const unsigned (&f)[32], uint32_t *wbase, int ws)
{
    uint32_t w[B];
    pack_unit<B>(f, w);
#pragma unroll
    for (int j = 0; j < B; ++j) wbase[j * ws] = w[j];
}
__device__ __forceinline__ void pack_store_b(int b, const unsigned (&f)[32], uint32_t *wbase, int ws)
{
    switch (b) {
    case 1: pack_store<1>(f, wbase, ws); break;
    case 2: pack_store<2>(f, wbase, ws); break;
    case 3: pack_store<3>(f, wbase, ws); break;
    case 4: pack_store<4>(f, wbase, ws); break;
    case 5: pack_store<5>(f, wbase, ws); break;
    case 6: pack_store<6>(f, wbase, ws); break;
    case 7: pack_store<7>(f, wbase, ws); break;
    case 8: pack_store<8>(f, wbase, ws); break;
    default: break;
    }
}

// hi part of the TF32 split of a finite value: nearest 11-bit significand, ties away (what cvt.rna.tf32 returns for finite
// inputs, without its NaN / infinity selects; the lo part a - hi is exact in fp32 either way)
__device__ __forceinline__ uint32_t tf32_near(float a) { return (__float_as_uint(a) + 0x1000u) & 0xffffe000u; }
__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }

static size_t tile_smem_bytes(int max_stride, int max_rows, bool cb_exact)
{
    return (size_t)kTile * kXsLd * 4 + (size_t)kTile * max_rows * 8 + 512 * 8 * (cb_exact ? 2 : 1) + 1024 * 4 +
           (size_t)kTile * max_rows * 2 + 16 + (size_t)kTile * max_rows * 4 + (size_t)kTile * kIdxLd + kMaxUnits * sizeof(UnitDesc) + kMaxFastItems * sizeof(FastItem) +
           16 + kMetaBytes + (size_t)kTileQueue * 2 + (size_t)max_stride + 64;
}

template <typename T>
__global__ void __launch_bounds__(kTileThreads, 1)
quantize_tile_kernel(const HeadMeta *__restrict__ metas, uint8_t *__restrict__ cache,
                     const T *__restrict__ k_new, const T *__restrict__ v_new, const double *__restrict__ cb64, int batch,
                     int n_new, int Hkv, const int32_t *__restrict__ seq_len, int64_t n_cap, int64_t max_tokens,
                     int cb_exact, int max_rows, const float2 *__restrict__ rot_hl)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int h = blockIdx.y % Hkv, lrel = blockIdx.y / Hkv, s = blockIdx.z;
#if BGTQ_APPEND_PHASES
    long long tph[10]; int nph = 0;
#define TPH() do { tph[nph++] = clock64(); } while (0)
#else
#define TPH() do { } while (0)
#endif
    TPH();
    const int64_t t0 = seq_len[s];
    const int64_t t_end = min(t0 + (int64_t)n_new, max_tokens);
    const int64_t tile = t0 / kTile + blockIdx.x;
    const int64_t tile_lo = tile * kTile;
    if (t0 > tile_lo || t_end < tile_lo + kTile) return;                  // not a whole tile of new tokens

    float *xs = reinterpret_cast<float *>(smem);                          // [128][kXsLd]: K in grouped order | V in grouped order
    double *sigma = reinterpret_cast<double *>(xs + kTile * kXsLd);       // [128][ns]
    double *tau = sigma + kTile * max_rows;                               // [512] (+ [512] V thresholds with exact-density codebooks)
    float *tau32 = reinterpret_cast<float *>(tau + (cb_exact ? 1024 : 512));   // [2][512]
    uint16_t *nrm = reinterpret_cast<uint16_t *>(tau32 + 1024);           // [128][ns]
    float *sig32 = reinterpret_cast<float *>(nrm + kTile * max_rows + 8);   // [128][ns]: (float)sigma, the fast path's scale
    uint8_t *idxs = reinterpret_cast<uint8_t *>(sig32 + kTile * max_rows);     // [128][kIdxLd]
    UnitDesc *units = reinterpret_cast<UnitDesc *>(idxs + kTile * kIdxLd);   // [32]
    FastItem *items = reinterpret_cast<FastItem *>(units + kMaxUnits);    // [32]
    int *cnt = reinterpret_cast<int *>(items + kMaxFastItems);            // [0] queue entries, [1] K items, [2] V items, [3] K units
    HeadMeta *Msp = reinterpret_cast<HeadMeta *>(cnt + 4);
    uint16_t *queue = reinterpret_cast<uint16_t *>(reinterpret_cast<unsigned char *>(Msp) + kMetaBytes);
    uint32_t *tbuf = reinterpret_cast<uint32_t *>(queue + kTileQueue);    // the tile, `stride` bytes (16-byte aligned)
    {
        const uint32_t *msrc = reinterpret_cast<const uint32_t *>(metas + blockIdx.y);
        uint32_t *mdst = reinterpret_cast<uint32_t *>(Msp);
        for (int i = tid; i < (int)(sizeof(HeadMeta) / 4); i += kTileThreads) mdst[i] = __ldg(msrc + i);
    }
    __syncthreads();
    const HeadMeta &M = *Msp;
    const int stride = M.tile_stride, ng = M.n_groups, kdim = M.kdim;
    const int nvg = M.n_vgroups, ns = ng + nvg;
    uint8_t *gtile = cache + n_cap * ((int64_t)batch * M.layer_prefix + (int64_t)s * M.layer_sum + M.head_prefix) + tile * stride;
    for (int i = tid; i < stride / 16; i += kTileThreads) reinterpret_cast<uint4 *>(tbuf)[i] = make_uint4(0, 0, 0, 0);
    const double *cbK = cb64 + (cb_exact ? (size_t)blockIdx.y * 1024 : 0);
    for (int i = tid; i < 511; i += kTileThreads) tau[i] = __dmul_rn(__dadd_rn(cbK[i], cbK[i + 1 < 511 ? i + 1 : i]), 0.5);
    if (cb_exact) {
        const double *cbV = cbK + 512;
        for (int i = tid; i < 511; i += kTileThreads) tau[512 + i] = __dmul_rn(__dadd_rn(cbV[i], cbV[i + 1 < 511 ? i + 1 : i]), 0.5);
    }
    const double *tauV = cb_exact ? tau + 512 : tau;
    if (tid == 0) {
        int n = 0, j = 0;
        for (int ks = 0; ks < M.n_ksteps; ++ks) {
            const KStep &K = M.ksteps[ks];
            const int g = K.flags >> 4;
            if (K.flags & 1) j = 0;
            units[n++] = UnitDesc{K.off0, K.b, K.nc0, (uint16_t)(M.gstart[g] + 8 * j), 0};
            ++j;
            if (K.off1 != 0xFFFF) { units[n++] = UnitDesc{K.off1, K.b, K.nc1, (uint16_t)(M.gstart[g] + 8 * j), 0}; ++j; }
        }
        cnt[3] = n;
        int ni = 0;
        for (int g = 0; g < ng; ++g)
            for (int n0 = 0; n0 < M.gm[g]; n0 += 16) items[ni++] = FastItem{M.gstart[g], (uint8_t)M.gm[g], (uint8_t)n0, M.gb[g], (uint8_t)g, 0, 0};
        cnt[1] = ni;
        for (int gv = 0; gv < nvg; ++gv)
            for (int n0 = 0; n0 < 16 * M.vgcnt[gv]; n0 += 16)
                items[ni++] = FastItem{(uint16_t)(128 + 16 * M.vgstart[gv]), (uint8_t)(16 * M.vgcnt[gv]), (uint8_t)n0, M.vgb[gv], (uint8_t)(ng + gv), 1, 0};
        cnt[2] = ni - cnt[1];
        cnt[0] = 0;
    }
    TPH();
    // ---- 1. gather: thread (column c = tid & 255, token half tid >> 8); inputs are fp32 / bf16 values, exact in fp32
    {
        const int col = tid & 255, th = tid >> 8;
        const T *g_src = col >= 128 ? v_new : k_new;
        const int g_off = col >= 128 ? 16 * M.vblk[(col - 128) >> 4] + (col & 15) : (col < kdim ? (int)M.coords[col] : -1);
        const int64_t rstep = (int64_t)Hkv * kDh;
        const int64_t row0 = ((((int64_t)lrel * batch + s) * n_new + (tile_lo - t0)) * Hkv + h) * kDh + (int64_t)th * 64 * rstep;
        float *xcol = xs + (size_t)th * 64 * kXsLd + col;
        if (g_off >= 0) {
#pragma unroll 1
            for (int t8 = 0; t8 < 64; t8 += 32) {                  // 32 independent loads in flight per thread
                T tv[32];
#pragma unroll
                for (int tt = 0; tt < 32; ++tt) tv[tt] = g_src[row0 + (t8 + tt) * rstep + g_off];
#pragma unroll
                for (int tt = 0; tt < 32; ++tt) xcol[(t8 + tt) * kXsLd] = to_f32(tv[tt]);
            }
        } else {
            for (int tt = 0; tt < 64; ++tt) xcol[tt * kXsLd] = 0.f;
        }
    }
    __syncthreads();
    TPH();
    for (int i = tid; i < 1022; i += kTileThreads) tau32[i + (i >= 511 ? 1 : 0)] = (float)(i < 511 ? tau[i] : tauV[i - 511]);
    // ---- 2. radii (exact fp64 chains in oracle order).  The long V chains go first, one per thread of the low warps; the
    //      second round is dealt from the other end so that no thread gets two long chains.
    {
        const int total = kTile * ns, nv = kTile * nvg;
        int w = tid;
        for (int r = 0; w < total; ++r, w = kTileThreads * r + ((r & 1) ? kTileThreads - 1 - tid : tid)) {
            int tt, g;
            if (w < nv) { tt = w / nvg; g = ng + w % nvg; } else { tt = (w - nv) / ng; g = (w - nv) % ng; }
            const int x0 = g < ng ? M.gstart[g] : 128 + 16 * M.vgstart[g - ng], m = g < ng ? M.gm[g] : 16 * M.vgcnt[g - ng];
            const float *x = xs + tt * kXsLd + x0;
            double ss = 0.0;
            for (int j = 0; j < m; ++j) { const double xv = (double)x[j]; ss = __fma_rn(xv, xv, ss); }
            const double r2 = __dsqrt_rn(ss);
            const double sgd = __ddiv_rn(r2, __dsqrt_rn((double)m));
            sigma[tt * ns + g] = sgd;
            sig32[tt * ns + g] = (float)sgd;
            uint16_t hb = __half_as_ushort(__double2half(r2));
            if (r2 >= 65520.0) hb = 0x7BFF;
            nrm[tt * ns + g] = hb;
        }
    }
    __syncthreads();
    TPH();
    // ---- 3. z ~ X Pi^T on the tensor cores and the threshold search.  Work unit = (item: 16 outputs of one rotation group,
    //      half: 4 m-tiles = 64 tokens); V units (m = 128, the long ones) are dealt first.
    {
        const int fg = lane >> 2, fc = lane & 3;
        const int nki = cnt[1], nvi = cnt[2], n_work = 2 * (nki + nvi);
#if BGTQ_APPEND_PHASES
        long long tmma = 0, tq = 0; int nun = 0;
#endif
        for (int u = warp; u < n_work; u += kTileWarps) {
#if BGTQ_APPEND_PHASES
            const long long ts0 = clock64(); ++nun;
#endif
            const int item = u < 2 * nvi ? nki + (u >> 1) : ((u - 2 * nvi) >> 1), half = u & 1;
            const FastItem it = items[item];
            const int m = it.m, nA = it.n0 + fg, nB = nA + 8;
            const bool two = it.n0 + 8 < m;
            const float2 *pA = rot_hl + rot_offset(m) + (size_t)(nA < m ? nA : 0) * m + fc;
            const float2 *pB = rot_hl + rot_offset(m) + (size_t)(nB < m ? nB : 0) * m + fc;
            const float *px = xs + (size_t)(half * 64 + fg) * kXsLd + it.x0 + fc;
            float acc[4][2][4];
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                for (int e = 0; e < 4; ++e) acc[mt][0][e] = acc[mt][1][e] = 0.f;
            // (the three products of an accumulator are issued eight MMAs apart -- term by term over the four m-tiles and two
            //  n-tiles -- so that no MMA waits for the one issued just before it)
            auto kstep = [&](const float2 ca0, const float2 ca1, const float2 cb0, const float2 cb1, int k0, bool va, bool vb) {
                uint32_t ah[4][4], al[4][4];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    const float *pm = px + mt * 16 * kXsLd + k0;
                    const float a[4] = {va ? pm[0] : 0.f, va ? pm[8 * kXsLd] : 0.f, vb ? pm[4] : 0.f, vb ? pm[8 * kXsLd + 4] : 0.f};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        ah[mt][e] = tf32_near(a[e]);
                        al[mt][e] = __float_as_uint(a[e] - __uint_as_float(ah[mt][e]));
                    }
                }
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {                                   // small terms first
                    mma_tf32(acc[mt][0], al[mt], __float_as_uint(ca0.x), __float_as_uint(ca1.x));
                    if (two) mma_tf32(acc[mt][1], al[mt], __float_as_uint(cb0.x), __float_as_uint(cb1.x));
                }
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    mma_tf32(acc[mt][0], ah[mt], __float_as_uint(ca0.y), __float_as_uint(ca1.y));
                    if (two) mma_tf32(acc[mt][1], ah[mt], __float_as_uint(cb0.y), __float_as_uint(cb1.y));
                }
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    mma_tf32(acc[mt][0], ah[mt], __float_as_uint(ca0.x), __float_as_uint(ca1.x));
                    if (two) mma_tf32(acc[mt][1], ah[mt], __float_as_uint(cb0.x), __float_as_uint(cb1.x));
                }
            };
            const int kfull = m & ~7;
#pragma unroll 4
            for (int k0 = 0; k0 < kfull; k0 += 8)                  // (unrolled: the operand loads of four k-steps are in flight together)
                kstep(__ldg(pA + k0), __ldg(pA + k0 + 4), __ldg(pB + k0), __ldg(pB + k0 + 4), k0, true, true);
            if (kfull < m) {                                   // ragged tail: k >= m contributes zero
                const bool va = kfull + fc < m, vb = kfull + fc + 4 < m;
                const float2 zero2 = make_float2(0.f, 0.f);
                kstep(va ? __ldg(pA + kfull) : zero2, vb ? __ldg(pA + kfull + 4) : zero2,
                      va ? __ldg(pB + kfull) : zero2, vb ? __ldg(pB + kfull + 4) : zero2, kfull, va, vb);
            }
#if BGTQ_APPEND_PHASES
            const long long ts1 = clock64(); tmma += ts1 - ts0;
#endif
            // codes from z where it is clear of the neighbouring thresholds; the rest go to the queue
            const float *tb = tau32 + (it.isv ? 512 : 0) + ((1 << it.b) - 1);
            const float gc = fast_guard(it.m);
            // Bisection over the 2^b - 1 thresholds, the eight codes of a lane side by side.  Both neighbours of the final
            // code are among the probed thresholds (the last probe that succeeded, the last that failed), so the smallest
            // |z - tau sigma| over the probes is the distance to the nearest neighbour: one running minimum replaces the
            // two extra look-ups of the sub-batch kernel (it can only flag more codes, never fewer).
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int ttA = half * 64 + mt * 16 + fg;                         // token rows ttA and ttA + 8
                const float sgA = sig32[ttA * ns + it.sidx], sgB = sig32[(ttA + 8) * ns + it.sidx];
                uint8_t *ip = idxs + ttA * kIdxLd + it.x0 + it.n0 + 2 * fc;
                float z8[8], d8[8];
                int a8[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) { z8[e] = acc[mt][e >> 2][e & 3]; a8[e] = 0; d8[e] = 3.0e38f; }
                for (int bit = it.b - 1; bit >= 0; --bit) {
                    const int step = 1 << bit;
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float t = tb[a8[e] + step - 1] * (((e >> 1) & 1) ? sgB : sgA);
                        d8[e] = fminf(d8[e], fabsf(z8[e] - t));
                        if (z8[e] > t) a8[e] += step;
                    }
                }
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int nl = it.n0 + 8 * (e >> 2) + 2 * fc + (e & 1);
                    if (nl >= it.m) continue;
                    ip[((e >> 1) & 1) * 8 * kIdxLd + 8 * (e >> 2) + (e & 1)] = (uint8_t)a8[e];
                    if (!(d8[e] > gc * (((e >> 1) & 1) ? sgB : sgA))) {
                        const int pos = atomicAdd(&cnt[0], 1);
                        if (pos < kTileQueue) queue[pos] = (uint16_t)(((ttA + 8 * ((e >> 1) & 1)) << 8) | (it.x0 + nl));
                    }
                }
            }
#if BGTQ_APPEND_PHASES
            tq += clock64() - ts1;
#endif
        }
#if BGTQ_APPEND_PHASES
        if ((tid == 0 || tid == 300) && blockIdx.x == 3 && blockIdx.y == 0 && blockIdx.z == 0)
            printf("tile phase 3 (tid %d): units %d mma %lld quant %lld\n", tid, nun, tmma, tq);
#endif
    }
    __syncthreads();
    TPH();
    // ---- 4. the exact fp64 chain (oracle order) for the queued (token, column) pairs
    {
        auto exact_code = [&](int tt, int col) {
            int m, x0, sidx, b;
            const double *tb;
            if (col >= 128) {
                const int gv = M.vbg[(col - 128) >> 4];
                m = 16 * M.vgcnt[gv]; x0 = 128 + 16 * M.vgstart[gv]; sidx = ng + gv; b = M.vgb[gv]; tb = tauV + ((1 << b) - 1);
            } else {
                int g = 0;
                while (g + 1 < ng && col >= M.gstart[g + 1]) ++g;
                m = M.gm[g]; x0 = M.gstart[g]; sidx = g; b = M.gb[g]; tb = tau + ((1 << b) - 1);
            }
            const float4 *Rq = reinterpret_cast<const float4 *>(rot_hl + rot_offset(m) + (size_t)(col - x0) * m);
            const float *x = xs + tt * kXsLd + x0;
            double zz = 0.0;
            int k = 0;
            for (; k + 32 <= m; k += 32) {
                float4 pf[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) pf[u] = __ldg(Rq + (k >> 1) + u);
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    zz = __fma_rn((double)(pf[u].x + pf[u].y), (double)x[k + 2 * u], zz);
                    zz = __fma_rn((double)(pf[u].z + pf[u].w), (double)x[k + 2 * u + 1], zz);
                }
            }
            for (; k < m; k += 2) {
                const float4 p = __ldg(Rq + (k >> 1));
                zz = __fma_rn((double)(p.x + p.y), (double)x[k], zz);
                zz = __fma_rn((double)(p.z + p.w), (double)x[k + 1], zz);
            }
            const double sg = sigma[tt * ns + sidx];
            int a = 0;
            for (int bit = b - 1; bit >= 0; --bit)
                if (zz > __dmul_rn(tb[a + (1 << bit) - 1], sg)) a += 1 << bit;
            idxs[tt * kIdxLd + col] = (uint8_t)a;
        };
        const int qn = cnt[0];
        if (qn <= kTileQueue) {
            for (int e = tid; e < qn; e += kTileThreads) exact_code(queue[e] >> 8, queue[e] & 255);
        } else {                                               // (queue overflow: never seen; every code takes the exact chain)
            for (int e = tid; e < kTile * 256; e += kTileThreads) {
                const int tt = e >> 8, col = e & 255;
                if (col >= 128 || col < kdim) exact_code(tt, col);
            }
        }
    }
    __syncthreads();
    TPH();
    // ---- 5. pack: one owner per (unit, lane); its eight four-slot groups (one per m-tile) in turn
    {
        const int kitems = cnt[3] * 32;
        for (int itx = tid; itx < kitems + 16 * 32; itx += kTileThreads) {
            if (itx < kitems) {
                const UnitDesc U = units[itx >> 5];
                const int lp = itx & 31, lanes = 8 * U.nc;
                if (lp >= lanes) continue;
                const int g8 = U.nc == 4 ? lp >> 2 : (U.nc == 2 ? lp >> 1 : (U.nc == 1 ? lp : (lp * 11) >> 5)), c = lp - g8 * U.nc;
                uint32_t *wbase = tbuf + (U.off >> 2) + lp;
                unsigned f[32];
#pragma unroll
                for (int k = 0; k < 32; ++k)                         // slot 4i + 2p + q: token 16i + 8p + g8, coordinate 2c + q
                    f[k] = idxs[(16 * (k >> 2) + 8 * ((k >> 1) & 1) + g8) * kIdxLd + U.ustart + 2 * c + (k & 1)];
                pack_store_b(U.b, f, wbase, lanes);
            } else {
                const int v = itx - kitems, unit = v >> 5, ln = v & 31;    // unit = 2J' + rho, J' = grouped V block
                const int gq = ln >> 2, c = ln & 3;
                const int u = 16 * (unit >> 1) + 8 * (unit & 1) + gq;      // grouped V coordinate
                const int bw = M.vbw[unit >> 1];
                uint32_t *wbase = tbuf + ((M.vboff[unit >> 1] + (unit & 1) * 128 * bw) >> 2) + ln;
                unsigned f[32];
#pragma unroll
                for (int k = 0; k < 32; ++k)                         // slot 4i + 2o + e: token 16i + 8o + 2c + e
                    f[k] = idxs[(16 * (k >> 2) + 8 * ((k >> 1) & 1) + 2 * c + (k & 1)) * kIdxLd + 128 + u];
                pack_store_b(bw, f, wbase, 32);
            }
        }
        for (int w = tid; w < kTile * ns; w += kTileThreads) {   // fp16 norms: token t at entry (t&7)*16 + (t>>4)*2 + ((t>>3)&1)
            const int t128 = w / ns, g = w % ns;
            const int slot = (t128 & 7) * 16 + (t128 >> 4) * 2 + ((t128 >> 3) & 1);
            const int off = g < ng ? M.knorm_off + 256 * g : M.vnorm_off + 256 * (g - ng);
            reinterpret_cast<uint16_t *>(reinterpret_cast<uint8_t *>(tbuf) + off)[slot] = nrm[t128 * ns + g];
        }
    }
    __syncthreads();
    TPH();
    {
        uint4 *dst = reinterpret_cast<uint4 *>(gtile);
        const uint4 *src = reinterpret_cast<const uint4 *>(tbuf);
        for (int i = tid; i < stride / 16; i += kTileThreads) dst[i] = src[i];
    }
    TPH();
#if BGTQ_APPEND_PHASES
    if ((tid == 0 || tid == 300) && blockIdx.x == 3 && blockIdx.y == 0 && blockIdx.z == 0)
        printf("tile phases (tid %d): setup %lld gather %lld radii %lld mma+quant %lld recheck(%d) %lld pack %lld writeback %lld\n", tid,
               tph[1] - tph[0], tph[2] - tph[1], tph[3] - tph[2], tph[4] - tph[3], cnt[0], tph[5] - tph[4], tph[6] - tph[5], tph[7] - tph[6]);
#endif
#undef TPH
}


__global__ void advance_seq_len_kernel(int32_t *seq_len, int batch, int n_new, int64_t max_tokens)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < batch) {
        int64_t v = (int64_t)seq_len[s] + n_new;
        seq_len[s] = (int32_t)(v > max_tokens ? max_tokens : v);
    }
}

static size_t append_smem_bytes(int max_stride, int max_rows, bool cb_exact = false, bool fast = false)
{
    return (size_t)kSub * 256 * 8 + 512 * 8 + kSub * max_rows * 8 + (kSub * max_rows + 8) * 2 + kSub * 256 +
           kMaxUnits * sizeof(UnitDesc) + 16 + kMetaBytes + (cb_exact ? 512 * 8 : 0) +
           (fast ? 1024 * 4 + kMaxFastItems * sizeof(FastItem) + kFastQueue * 2 + 16 : 0) + (size_t)max_stride + 64;
}

// Bulk appends (>= kFastMinTokens new tokens per sequence) take the tensor-core fast path; the decode-time append keeps the
// latency-shaped exact kernel.  Both write identical bytes.
constexpr int kFastMinTokens = 16;

int launch_quantize_append(const bgtq_layout *lay, int layer, int n_layers, void *cache, const void *k_new,
                           const void *v_new, int dt, int batch, int n_new, int32_t *seq_len,
                           int advance, int64_t max_tokens, const PageMap *pm, const RopeTab *rope, cudaStream_t st)
{
    const int64_t n_cap = (max_tokens + kTile - 1) / kTile;
    // The fast kernel runs 3 CTAs per SM (80 registers, 12 KB more shared memory), the exact one 4: a grid that fits one wave of
    // the exact kernel but not of the fast one would lose more to the second wave than the fast path gains (measured: 514
    // CTAs, 30 vs 39 G codes/s), so those grids keep the exact kernel.
    const int64_t n_cta = (int64_t)((n_new + kTile - 1) / kTile + 1) * lay->n_kv_heads * n_layers * batch;
    const bool fast = n_new >= kFastMinTokens && !append_exact_only() &&
                      (n_cta <= 3 * (int64_t)lay->sm_count || n_cta > 8 * (int64_t)lay->sm_count);
    const size_t smem = append_smem_bytes(lay->max_stride, lay->max_rows, lay->cb_exact != 0, fast);
    dim3 grid((n_new + kTile - 1) / kTile + 1, lay->n_kv_heads * n_layers, batch);
    // whole tiles of new tokens go to quantize_tile_kernel (one pass per tile); the sub-batch kernel keeps the partly
    // filled first / last tile of every sequence
    const size_t tsmem = tile_smem_bytes(lay->max_stride, lay->max_rows, lay->cb_exact != 0);
    const bool tiled = n_new >= kTile && !append_exact_only() && !pm && !rope && lay->format == 1 && tsmem <= 227 * 1024;
    const HeadMeta *metas = lay->d_meta + (size_t)layer * lay->n_kv_heads;
    if (first_use_on_device(1)) {   // once per device, outside any stream capture
        const int maxs = (int)append_smem_bytes(16 * kDh * 8 + 256 * 16 + 16 * kDh * 8, 16, true, true);
#define BGTQ_APPEND_ATTR(T, R, G) \
        CUDA_TRY(cudaFuncSetAttribute(quantize_append_kernel<T, R, G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxs)); \
        CUDA_TRY(cudaFuncSetAttribute(quantize_append_kernel<T, R, G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxs))
        BGTQ_APPEND_ATTR(float, false, false); BGTQ_APPEND_ATTR(__nv_bfloat16, false, false);
        BGTQ_APPEND_ATTR(float, true, false);  BGTQ_APPEND_ATTR(__nv_bfloat16, true, false);
        BGTQ_APPEND_ATTR(float, false, true);  BGTQ_APPEND_ATTR(__nv_bfloat16, false, true);
#undef BGTQ_APPEND_ATTR
        CUDA_TRY(cudaFuncSetAttribute(quantize_tile_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CUDA_TRY(cudaFuncSetAttribute(quantize_tile_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    }
    const int32_t *pt = pm ? pm->table : nullptr;
    const int pstride = pm ? pm->table_stride : 0;
    const int64_t n_pages = pm ? pm->n_pages : 0;
    const float *rc = rope ? rope->cos : nullptr, *rs = rope ? rope->sin : nullptr;
    // (a runtime `pages ? :` in the kernel costs 30 % of the bulk append rate, hence the template switch)
    if (pm && rope) { set_error("bgtq_quantize_append: paged + fused RoPE is not built"); return BGTQ_EINVAL; }
    auto launch = [&](auto plain, auto roped, auto paged, auto *kp, auto *vp) {
        auto kern = pm ? paged : (rope ? roped : plain);
        const double *cb = lay->cb_exact ? lay->d_hcb64 + (size_t)layer * lay->n_kv_heads * 1024 : lay->d_cb64;
        kern<<<grid, kAppendThreads, smem, st>>>(metas, (uint8_t *)cache, kp, vp, cb, lay->d_rot_t, batch, n_new,
                                                 lay->n_kv_heads, seq_len, n_cap, max_tokens, pt, pstride, n_pages, rc, rs,
                                                 lay->pairing, lay->cb_exact, lay->max_rows, lay->d_rot_hl, tiled ? 1 : 0);
    };
    if (tiled) {
        const double *cb = lay->cb_exact ? lay->d_hcb64 + (size_t)layer * lay->n_kv_heads * 1024 : lay->d_cb64;
        if (dt == BGTQ_F32)
            quantize_tile_kernel<float><<<grid, kTileThreads, tsmem, st>>>(metas, (uint8_t *)cache, (const float *)k_new, (const float *)v_new, cb, batch, n_new,
                                                                         lay->n_kv_heads, seq_len, n_cap, max_tokens, lay->cb_exact, lay->max_rows, lay->d_rot_hl);
        else
            quantize_tile_kernel<__nv_bfloat16><<<grid, kTileThreads, tsmem, st>>>(metas, (uint8_t *)cache, (const __nv_bfloat16 *)k_new, (const __nv_bfloat16 *)v_new, cb,
                                                                                 batch, n_new, lay->n_kv_heads, seq_len, n_cap, max_tokens, lay->cb_exact,
                                                                                 lay->max_rows, lay->d_rot_hl);
        count_launch();
        CUDA_TRY(cudaGetLastError());
    }
#define BGTQ_APPEND_LAUNCH(T, F) \
        launch(quantize_append_kernel<T, false, false, F>, quantize_append_kernel<T, true, false, F>, \
               quantize_append_kernel<T, false, true, F>, (const T *)k_new, (const T *)v_new)
    if (dt == BGTQ_F32) { if (fast) BGTQ_APPEND_LAUNCH(float, true); else BGTQ_APPEND_LAUNCH(float, false); }
    else { if (fast) BGTQ_APPEND_LAUNCH(__nv_bfloat16, true); else BGTQ_APPEND_LAUNCH(__nv_bfloat16, false); }
#undef BGTQ_APPEND_LAUNCH
    count_launch();
    CUDA_TRY(cudaGetLastError());
    if (advance) {
        advance_seq_len_kernel<<<(batch + 127) / 128, 128, 0, st>>>(seq_len, batch, n_new, max_tokens);
        count_launch();
        CUDA_TRY(cudaGetLastError());
    }
    return BGTQ_OK;
}

}  // namespace bgtq
