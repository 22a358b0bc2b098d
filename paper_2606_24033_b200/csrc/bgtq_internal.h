// bgtq_internal.h -- shared declarations of the library's translation units (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/bgtq.h"

namespace bgtq {

constexpr int kDh = 128;          // head dimension the kernels are written for
constexpr int kTile = 128;        // tokens per tile
constexpr int kMaxGroups = 8;
constexpr int kMaxKSteps = 16;    // sum_g ceil(m_g/16) <= 8 + 7

// One k16 step of the QK^T product: two half-step units (8 coordinates each) of one group.
struct KStep {
    uint16_t off0;     // byte offset of the first unit inside the tile
    uint16_t off1;     // second unit, 0xFFFF if the group ends after the first
    uint8_t b;         // code width of the group
    uint8_t nc0;       // lanes per 8-token row holding data in unit 0 (4 = full, 1..3 partial)
    uint8_t nc1;       // same for unit 1 (0 if absent)
    uint8_t flags;     // bit0 first step of its group, bit1 last step; bits 4..7 group index
};

// BGTQ-v2 (row order): one chunk = up to 32 grouped coordinates of one group, one token per lane.
struct Chunk2 {
    uint16_t off;      // byte offset of the chunk's first word plane inside a quadrant's K-code section
    uint16_t ustart;   // grouped-order coordinate of slot 0
    uint8_t b;         // code width
    uint8_t r;         // slots in use (even, 2..32)
    uint8_t nw;        // 32-bit words per lane
    uint8_t flags;     // bit0 first chunk of its group; bits 4..7 group index
};
constexpr int kMaxChunks = 12;    // sum_g ceil(m_g/32) <= 4 + 7

// Static layout metadata of one (layer, KV head)   ("static layout metadata")
struct HeadMeta {
    int32_t n_groups, kdim, n_ksteps, b_v;      // n_ksteps: k16 steps (v1) / chunks (v2)
    int32_t tile_stride, kcode_bytes, knorm_off, vnorm_off, vcode_off, format;   // format: 1 = BGTQ-v1, 2 = BGTQ-v2
    int64_t layer_prefix;   // sum of tile strides of all heads of all earlier layers
    int64_t layer_sum;      // sum of tile strides of the heads of this layer
    int64_t head_prefix;    // sum of tile strides of earlier heads of this layer
    int32_t goff[kMaxGroups];      // byte offset of the group's codes inside the tile
    uint16_t gm[kMaxGroups];       // coordinates in the group
    uint16_t gstart[kMaxGroups];   // first grouped-order coordinate of the group
    uint8_t gb[kMaxGroups];        // width of the group
    uint8_t coords[kDh];           // grouped order -> original coordinate (Q9)
    // V side (reading Q19): same-width groups of 16-coordinate V blocks, ascending width; a uniform V width is one group of
    // all 8 blocks.  "Grouped block" J' = position of a block in the grouped order (the order of the accumulator and of the
    // V code section); the tile holds one fp16 norm row per V group at vnorm_off + 256 * gv.
    uint8_t n_vgroups, vpad[3];
    uint8_t vgb[kMaxGroups];       // width of V group gv
    uint8_t vgcnt[kMaxGroups];     // blocks in the group (m = 16 * vgcnt)
    uint8_t vgstart[kMaxGroups];   // first grouped block of the group
    uint8_t vblk[kMaxGroups];      // grouped block -> original block (coordinates 16 * vblk .. + 15)
    uint8_t vbg[kMaxGroups];       // grouped block -> V group
    uint8_t vbw[kMaxGroups];       // grouped block -> width
    uint16_t vboff[kMaxGroups];    // grouped block -> byte offset of its first unit inside the tile
    union {
        KStep ksteps[kMaxKSteps];  // v1
        Chunk2 chunks[kMaxKSteps]; // v2 (kMaxChunks used); kcode_bytes = 4 * (bytes of one quadrant)
    };
};
static_assert(sizeof(KStep) == 8 && sizeof(Chunk2) == 8, "k-step / chunk descriptors are 8 bytes");
static_assert(kDh / 16 == kMaxGroups, "eight V blocks of 16 coordinates");

}  // namespace bgtq

struct bgtq_layout {
    int n_layers, n_kv_heads, n_q_heads, d_h, b_v, pairing;     // b_v: the uniform V width, 0 when widths come from bits_v
    int v_grouped;                        // 1 when some head has more than one V group (V-side allocator, reading Q19)
    int format;                           // 1 = BGTQ-v1 (fragment order), 2 = BGTQ-v2 (row order)
    uint8_t *d_planes;                    // v2: e4m3 byte planes of the codebooks, see codebook_planes()
    float kappa[9];                       // v2: plane scale of width b
    int max_stride;                       // largest tile stride over all heads
    int max_rows;                         // largest number of norm rows (K groups + V groups) over all heads
    int max_chunks;                       // v2: largest number of K chunks over all heads
    std::vector<bgtq::HeadMeta> meta;     // host copy, [layer][kv_head]
    int64_t total_stride_sum;             // sum of tile strides over all (layer, head)
    bgtq::HeadMeta *d_meta;               // device copy
    float *d_rot;                         // rotation table, row-major Pi^(m)[j][k]
    float *d_rot_t;                       // transposed: Pi^(m)[j][k] stored at [k][j]
    float2 *d_rot_hl;                     // row-major {tf32(Pi), Pi - tf32(Pi)}: operands of the append fast path
    uint16_t *d_cb16;                     // fp16 bits of the 511 codebook levels (C_b at 2^b-1)
    double *d_cb64;                       // same levels as fp64
    // exact-density codebooks (cb_exact = 1): one table set per (layer, kv head) -- groups and widths are
    // 1:1 inside a head, so the table of width w holds C_{w, m_g} of that head's group of width w; V uses C_{b_V, d_h}.
    int cb_exact;
    uint16_t *d_hcb16;                    // [head][2][kHeadLutHalves]: K, V: flat fp16 levels (512) + the 5-bit pair table (1024 x 2)
    double *d_hcb64;                      // [head][2][512]
    int sm_count;
};

namespace bgtq {

void set_error(const std::string &msg);
int cuda_fail(cudaError_t e, const char *what);
void count_launch(int n = 1);
// true exactly once per (key, current CUDA device): kernel function attributes are per device and must be set on each
// device the library is used on (thread-safe)
bool first_use_on_device(int key);
void codebook_levels(int b, double *levels);
// e4m3 byte planes of C_b (v2 decode path): level k of width b is represented as (hi[k] + lo[k]) / kappa with hi, lo
// e4m3 values; kappa in [32, 64] is chosen per width to minimise the largest relative error (0 for b = 1, 3; < 2e-6 for
// b = 2; < 2e-4 for b = 4; < 1.3e-3 for b >= 5).  hi, lo receive 2^b bytes each.
void codebook_planes(int b, float *kappa, uint8_t *hi, uint8_t *lo);
// exact-density codebook C_{b,m}: Lloyd-Max quantiser of the density of a coordinate of sqrt(m) x (uniform unit vector of
// R^m), rounded to fp16 (m even)
void codebook_levels_sphere(int b, int m, double *levels);
constexpr int kHeadLutHalves = 512 + 2048;
constexpr int kPlaneBytes = 2 * 512;   // [plane][flat level index (2^b - 1 + k)]

__host__ __device__ inline int64_t rot_offset(int m)  // element offset of Pi^(m), m even: sum of m'^2, m' = 2,4,..,m-2
{
    const int64_t n = m / 2;
    return 4 * ((n - 1) * n * (2 * n - 1) / 6);
}

// Paged cache (bgtq_*_paged): pools [layer][kv head][page], one page = one 128-token tile of that head;
// table[seq * table_stride + tile] = page index, the same index in every (layer, head) pool.  table == nullptr:
// the contiguous layout [layer][seq][kv head][tile].
struct PageMap {
    const int32_t *table;
    int table_stride;
    int64_t n_pages;
};

// Protected regime (bgtq_decode_attention_protected): fp16 windows [layer][seq][kv head][n_sink + n_recent][d_h]
struct Window {
    const void *k, *v;
    int n_sink, n_recent;
};

// RoPE fused into append (bgtq_quantize_append_rope): fp32 tables [rows][d_h/2], row = token position
struct RopeTab {
    const float *cos, *sin;
};

// implemented in the .cu files
int launch_block_energy(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt, int Hq,
                        int Hkv, int d_h, int pairing, int kind, float *scores, float *eq_out,
                        float *ek_out, void *ws, size_t ws_bytes, cudaStream_t st);
size_t block_energy_ws_bytes(int Hq, int Hkv, int d_h);
int launch_block_energy_static(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt, int Hq, int Hkv, int d_h,
                               int pairing, int kind, float *scores, float *eq_out, float *ek_out, cudaStream_t st);
int block_energy_static_max_row_elems();
int launch_v_block_energy(const void *v, int64_t n, int dt, int Hkv, int d_h, float *scores, void *ws, cudaStream_t st);
int launch_allocate(const float *scores, int n_heads, int L, int b_min, int b_max, int B,
                    uint8_t *bits, cudaStream_t st);
// test hook (bgtq_debug_append_exact_only): force the exact fp64 append kernel for bulk appends too
bool append_exact_only();
void set_append_exact_only(bool on);
int debug_decode_unit_exact(int b, int m, const uint32_t *words, float *values);
int launch_quantize_append(const bgtq_layout *lay, int layer, int n_layers, void *cache, const void *k_new,
                           const void *v_new, int dt, int batch, int n_new, int32_t *seq_len,
                           int advance, int64_t max_tokens, const PageMap *pm, const RopeTab *rope, cudaStream_t st);
int launch_decode(const bgtq_layout *lay, int layer0, int n_layers, const void *cache,
                  const void *q, const int32_t *seq_len, int batch, int64_t max_tokens,
                  float scale, void *out, void *ws, size_t ws_bytes, const PageMap *pm, cudaStream_t st,
                  const Window *win = nullptr);
int launch_window_append(const void *k_new, const void *v_new, int dt, int n_layers, int batch, int n_new, int Hkv,
                         const int32_t *seq_len, int64_t max_tokens, void *win_k, void *win_v, int n_sink, int n_recent,
                         cudaStream_t st);
size_t decode_ws_bytes(const bgtq_layout *lay, int batch, int n_layers);
int launch_decode2(const bgtq_layout *lay, int layer0, int n_layers, const void *cache,
                   const void *q, const int32_t *seq_len, int batch, int64_t max_tokens,
                   float scale, void *out, void *ws, size_t ws_bytes, const PageMap *pm, cudaStream_t st,
                   const Window *win = nullptr);
size_t decode2_ws_bytes(const bgtq_layout *lay, int batch, int n_layers);
int debug_decode_unit(int b, const uint32_t *words, float *values);
size_t prefill_ws_bytes(const bgtq_layout *lay, int batch, int n_q);
int launch_prefill(const bgtq_layout *lay, int layer, const void *cache, const void *q, const int32_t *seq_len,
                   int batch, int n_q, int64_t max_tokens, float scale, void *out, void *ws, size_t ws_bytes,
                   cudaStream_t st);
size_t fp16_ws_bytes(int sm_count, int batch, int n_layers, int Hkv);
int launch_fp16_decode(int n_layers, int batch, int Hq, int Hkv, const void *k_cache, const void *v_cache,
                       const void *q, const int32_t *seq_len, int64_t max_tokens, float scale, void *out,
                       void *ws, size_t ws_bytes, cudaStream_t st);
const char *microbench_name(int which);
int microbench_run(int which, int warps, double *value);
void profile_decode_enable(int enable);
int profile_decode_read(double *ms_sum, int *count);

}  // namespace bgtq
