/*
 * bgtq.h -- C-ABI of the B200-native Block-GTQ packed-cache decode path.
 *
 * Paper: "RoPE-Aware Bit Allocation for KV-Cache Quantization" (arxiv/paper_2606_24033);
 * citations are PAPER.md:<line>; "Qn" are the readings listed in DESIGN.md section 2.
 *
 * Conventions (all entry points):
 *   - return value is a bgtq_status (0 = ok, <0 = error); nothing throws or aborts;
 *     bgtq_last_error() returns a thread-local description of the last failure.
 *   - pointers marked [device] are CUDA device pointers owned by the caller (PyTorch owns the
 *     memory); pointers marked [host] are plain host memory.  The library allocates device memory
 *     only inside bgtq_layout_create (small static metadata) and frees it in bgtq_layout_destroy.
 *   - device work is asynchronous on the caller's `stream` (a cudaStream_t passed as void*;
 *     NULL = default stream).  No hidden synchronisation.
 *   - tensors are dense row-major with the listed shapes.  K and q are POST-RoPE (the paper
 *     quantises after rotary), so no positions cross this boundary.
 *   - GQA map: query head a uses KV head a / (n_q_heads / n_kv_heads)   (Q18).
 *   - there is no CPU fallback: every device entry point needs an sm_100a GPU.
 */
#ifndef BGTQ_H
#define BGTQ_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BGTQ_OK = 0,
    BGTQ_EINVAL = -1,     /* bad argument (shape, enum, null pointer, negative/NaN score) */
    BGTQ_EBUDGET = -2,    /* B not in [L*b_min, L*b_max] */
    BGTQ_ECAPACITY = -3,  /* n_new or batch exceeds what the cache was sized for */
    BGTQ_EWORKSPACE = -4, /* workspace too small */
    BGTQ_ECUDA = -5       /* a CUDA runtime call failed */
} bgtq_status;

typedef enum { BGTQ_F32 = 0, BGTQ_BF16 = 1 } bgtq_dtype;
/* which coordinates form RoPE block i (Q1): HALF = (i, i+d_h/2), INTERLEAVED = (2i, 2i+1) */
typedef enum { BGTQ_PAIR_HALF = 0, BGTQ_PAIR_INTERLEAVED = 1 } bgtq_pairing;
/* score kinds; QK_AVG is Eq. 1 / Eq. 4 */
typedef enum { BGTQ_QK_AVG = 0, BGTQ_QK_MAX = 1, BGTQ_QK_PRODUCT = 2, BGTQ_K_ONLY = 3,
               BGTQ_Q_ONLY = 4 } bgtq_score;

#define BGTQ_TILE_TOKENS 128   /* tokens per packed tile */
#define BGTQ_MAX_WIDTH 8       /* widest code, bits per coordinate */

const char *bgtq_last_error(void);

/* TQ-MSE scalar codebook C_b (Q7): the 2^b levels of the Lloyd-Max quantiser of N(0,1),
 * ascending, symmetric, rounded to fp16-representable values; b = 0 is {0}.  PAPER.md:49, 114.
 * levels [host] receives 2^b floats.  Computed by the library itself (csrc/codebook.cpp). */
int bgtq_codebook(int b, float *levels);

/* ---- a1: block-energy score, Eq. 1 = Eq. 4, Alg. 2.
 *   Eq[h][i] = 1/(n_q*G) sum_t sum_{g in G(h)} (q[t][g][a(i)]^2 + q[t][g][b(i)]^2)   (square, then mean)
 *   Ek[h][i] = 1/n_k     sum_t               (k[t][h][a(i)]^2 + k[t][h][b(i)]^2)
 *   scores[h][i] = kind(Eq, Ek);  QK_AVG = (Eq+Ek)/2.  n_q and n_k are independent (Q15).
 * q [device] [n_q, n_q_heads, d_h], k [device] [n_k, n_kv_heads, d_h], both of dtype `dt`.
 * scores [device] float [n_kv_heads, d_h/2]; eq_out / ek_out [device] same shape, may be NULL.
 * workspace [device], at least bgtq_block_energy_workspace_bytes(...) bytes; contents scratch.
 * Deterministic (fixed reduction order).  One layer per call, ONE kernel launch (a cooperative launch: a grid-wide
 * barrier separates the streaming pass from the fp64 reduction; needs a device with cooperative-launch support). */
size_t bgtq_block_energy_workspace_bytes(int n_q_heads, int n_kv_heads, int d_h);
int bgtq_block_energy(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt,
                      int n_q_heads, int n_kv_heads, int d_h, int pairing, int kind,
                      float *scores, float *eq_out, float *ek_out,
                      void *workspace, size_t workspace_bytes, void *stream);

/* The same computation for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no workspace argument -- the partial sums live in a file-scope device array of
 * the library, 4 MiB per GPU that loads the library, held until the process exits.  The call allocates nothing (no
 * cudaMalloc / cudaFree, no allocating library routine); the array's device address is looked up once per device.
 * Limit: (n_q_heads + n_kv_heads) * d_h <= bgtq_block_energy_static_max_row_elems() = 8192 (e.g. 48 + 16 heads at
 * d_h = 128); beyond it the call returns BGTQ_EWORKSPACE and launches nothing -- use bgtq_block_energy.  n_q, n_k are
 * not limited.  Token chunks are capped at 128 per tensor (workspace path: 512), so fp32 partial sums group differently:
 * results agree with bgtq_block_energy to ~1e-6 relative, not bit for bit.  Deterministic.
 * ALL calls share the one array (it keeps the last call's contents; nothing in it needs clearing, a call reads only what
 * it has written): calls that overlap on the GPU -- other streams, concurrently replayed graphs, several host threads on
 * one device -- RACE.  Serialise them (one stream) or use bgtq_block_energy with a workspace per call. */
int bgtq_block_energy_static_max_row_elems(void);
int bgtq_block_energy_static(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt,
                             int n_q_heads, int n_kv_heads, int d_h, int pairing, int kind,
                             float *scores, float *eq_out, float *ek_out, void *stream);

/* ---- a2: greedy marginal-gain allocation, Alg. 1, optimal by Thm. 1.
 * Per head: b_i = b_min; repeat B - L*b_min times: give one bit to the block with the largest
 * Delta_i = 3/4 * s_i * 4^-b_i among those with b_i < b_max; ties -> smallest i (Q4).
 * scores float [n_heads, n_blocks]; bits uint8 [n_heads, n_blocks], sum_i bits = total_bits_B.
 * on_device = 0: both pointers [host], runs on the calling thread (stream ignored; negative or
 *   NaN scores -> BGTQ_EINVAL).  on_device = 1: both [device], one warp per head, asynchronous
 *   (a negative/NaN score is treated as 0 there). */
int bgtq_allocate(const float *scores, int n_heads, int n_blocks, int b_min, int b_max,
                  int total_bits_B, uint8_t *bits, int on_device, void *stream);

/* ---- a3: same-width grouping -> static layout metadata.
 * bits [host] uint8 [n_layers, n_kv_heads, d_h/2] (widths 0..8; width 0 = block not stored,
 *   decodes to 0, Q3).  Groups G_w = {i : bits_i = w}, w ascending; coordinates inside a group
 *   [a(i1), b(i1), a(i2), ...] (Q9).  b_v: uniform V width (1..8).
 * rotations [host] float: the TQ-MSE rotation table (Q8), Pi^(m) for m = 2,4,..,d_h,
 *   row-major Pi^(m)[j][k] at offset sum_{m'<m, m' even} m'^2 + j*m + k.  It is a random draw of the
 *   method and therefore an INPUT (data), copied to the device.
 * The physical format is "BGTQ-v1": tile of 128 tokens =
 *   [K codes | K norms (fp16) per group | V norms (fp16) | V codes], no padding;
 *   bytes per token = 16*bbar_K + 16*b_V + 2*(n_groups+1) at d_h = 128.
 * d_h must be 128.  The layout owns a few hundred KB of device memory. */
typedef struct bgtq_layout bgtq_layout;
int bgtq_layout_create(const uint8_t *bits, int n_layers, int n_kv_heads, int n_q_heads, int d_h,
                       int b_v, int pairing, const float *rotations, bgtq_layout **out);
/* The same with an explicit physical format ("static layout metadata"; DESIGN.md sections 4, 4b):
 *   BGTQ_FORMAT_V1  "fragment order": code words follow the mma.sync fragment order of the round-1 decode kernel;
 *                   no padding (16*bbar_K + 16*b_V + 2*(n_groups+1) bytes per token at d_h = 128).
 *   BGTQ_FORMAT_V2  "row order": a code word belongs to ONE operand row (a token for K, a dimension for V), so the
 *                   decode kernel can write unpacked 8-bit operand rows straight into tensor memory for tcgen05.mma.
 *                   K groups are stored in chunks of <= 32 coordinates per token, each chunk rounded up to whole 32-bit
 *                   words (same bytes as V1 when every group holds a multiple of 32 coordinates).
 * Every call below works on either format unless stated otherwise; the cache bytes of the two formats differ. */
typedef enum { BGTQ_FORMAT_V1 = 1, BGTQ_FORMAT_V2 = 2 } bgtq_format;
/* OR-ed into `format`: exact-density TQ-MSE codebooks (reading Q7b in DESIGN.md).  PAPER.md:49 scalar-
 * quantises the rotated coordinates of a NORMALISED vector; a coordinate of sqrt(m) x (uniform unit vector of R^m) has the
 * density ~ (1 - x^2/m)^((m-3)/2), not N(0,1).  With this flag the group of m coordinates at width b uses C_{b,m}, the
 * Lloyd-Max quantiser of that density (fp16-rounded; bgtq_codebook_exact), V uses C_{b_V, d_h}; without it every group
 * shares C_b = bgtq_codebook(b) (Q7).  Supported by BGTQ_FORMAT_V1: append (all variants), decode attention (contiguous
 * and protected); prefill, the paged decode and BGTQ_FORMAT_V2 return BGTQ_EINVAL. */
#define BGTQ_CODEBOOK_EXACT 0x100
int bgtq_codebook_exact(int b, int m, float *levels);
int bgtq_layout_create_format(const uint8_t *bits, int n_layers, int n_kv_heads, int n_q_heads, int d_h,
                              int b_v, int pairing, const float *rotations, int format, bgtq_layout **out);
int bgtq_layout_format(const bgtq_layout *layout);

/* ---- V-side allocator ("Adding a V-side allocator to Block-GTQ is a natural extension",
 * PAPER.md:318; the paper gives no construction, reading Q19 is the one built here).
 * A V block is BGTQ_V_BLOCK = 16 consecutive coordinates of the head (d_h/16 blocks).  Its score is the mean squared block
 * norm  s^V[h][j] = 1/n sum_t sum_{u<16} v[t][h][16j+u]^2  (bgtq_v_block_energy): by the TQ-MSE rate law
 * the squared error block j adds to an attention output is proportional to s^V_j 4^-b_j, the objective Alg. 1 minimises,
 * so the widths come from bgtq_allocate(scores = s^V, n_blocks = d_h/16, B = bbar_V * d_h/16).  Blocks of equal width form
 * one V group (ascending width, member blocks ascending), encoded by one TQ-MSE encoder with rotation Pi^(m), m = 16 x
 * blocks, and one fp16 norm per (token, V group) -- exactly what PAPER.md:108 does for K.
 *   v [device] [n, n_kv_heads, d_h] of dtype dt; scores [device] float [n_kv_heads, d_h/16]; workspace [device] scratch of
 *   at least bgtq_v_block_energy_workspace_bytes bytes.  Deterministic.  One layer per call.
 * bgtq_layout_create_kv: bits_k as `bits` of bgtq_layout_create; bits_v [host] uint8 [n_layers, n_kv_heads, d_h/16], widths
 *   1..8 (every V block is stored).  Tile = [K codes | K norms | V norms: one row per V group | V codes: groups in order,
 *   two units of 128*w bytes per block]; all widths of a head equal = the uniform layout, byte for byte (heads may then
 *   still differ from each other).  BGTQ_FORMAT_V1 only (BGTQ_CODEBOOK_EXACT may be OR-ed in: V group (w, m) uses C_{w,m}).
 *   Heads with more than one V group are served by append (all variants) and decode attention (contiguous and protected);
 *   bgtq_prefill_attention and bgtq_decode_attention_paged return BGTQ_EINVAL for such a layout. */
#define BGTQ_V_BLOCK 16
size_t bgtq_v_block_energy_workspace_bytes(int n_kv_heads, int d_h);
int bgtq_v_block_energy(const void *v, int64_t n, int dt, int n_kv_heads, int d_h, float *scores,
                        void *workspace, size_t workspace_bytes, void *stream);
int bgtq_layout_create_kv(const uint8_t *bits_k, const uint8_t *bits_v, int n_layers, int n_kv_heads, int n_q_heads,
                          int d_h, int pairing, const float *rotations, int format, bgtq_layout **out);
void bgtq_layout_destroy(bgtq_layout *layout);

/* Sizes.  cache: one buffer for all layers, order [layer][sequence][head][tile], which the CALLER
 * allocates and ZERO-INITIALISES once (cudaMemset); max_tokens is the per-sequence capacity
 * (rounded up to whole tiles).  token_bytes: tile stride / 128 of (layer, kv_head) -- the
 * roofline input.  workspace: scratch for bgtq_decode_attention (n_layers_per_call = 1 for the
 * per-layer call). */
size_t bgtq_cache_bytes(const bgtq_layout *layout, int batch, int64_t max_tokens);
double bgtq_token_bytes(const bgtq_layout *layout, int layer, int kv_head);
size_t bgtq_workspace_bytes(const bgtq_layout *layout, int batch, int n_layers_per_call);
/* byte offset of the packed region of (layer, sequence, kv_head) inside the cache, and its tile
 * stride; for tests and tools that compare regions with the oracle's packer. */
int64_t bgtq_region_offset(const bgtq_layout *layout, int layer, int seq, int kv_head, int batch,
                           int64_t max_tokens);
int64_t bgtq_tile_stride(const bgtq_layout *layout, int layer, int kv_head);

/* ---- a4: quantize-on-append.  TQ-MSE per same-width K group and for
 * V as one group; code streams + fp16 norms written in the layout the decode kernel reads
 * (PAPER.md:112, 122).  The result is the exact fp64 sequence of DESIGN.md section 3 (codes, norms and
 * bytes are bit-exact against the oracle).  A call with fewer than 16 new tokens per sequence evaluates that
 * sequence directly; a bulk append evaluates the rotation on the tensor cores (TF32, hi/lo split) and
 * recomputes with the exact fp64 chain every code whose rotated value lies within a guard band of a
 * quantisation threshold -- the same bytes, checked against the exact kernel (bgtq_debug_append_exact_only).
 * Within a bulk append every tile whose 128 tokens are all new is quantised in one pass by one CTA
 * (quantize_tile_kernel; contiguous BGTQ-v1 caches, post-RoPE keys); the partly filled first / last tile of a
 * sequence, paged caches, fused RoPE and BGTQ-v2 take the 16-token sub-batch kernel.  One call may therefore launch two
 * kernels on `stream`; they touch disjoint tiles.
 * k_new, v_new [device] [batch, n_new, n_kv_heads, d_h] of dtype dt (post-RoPE K).
 * seq_len [device] int32 [batch]: tokens already cached; sequence s receives its n_new tokens at
 *   positions seq_len[s] .. seq_len[s]+n_new-1 and, if advance_seq_len != 0, seq_len[s] is advanced
 *   by n_new (by a kernel on `stream`; a model appends to every layer with the same seq_len and
 *   advances on the last).  Tokens at positions >= max_tokens (the caller's capacity, NOT rounded up to
 *   a whole tile) are dropped and seq_len saturates at max_tokens (BGTQ_ECAPACITY if n_new > max_tokens
 *   is detectable on the host).
 * Only the fields of the new tokens change.  One layer per call. */
int bgtq_quantize_append(const bgtq_layout *layout, int layer, void *cache, const void *k_new,
                         const void *v_new, int dt, int batch, int n_new, int32_t *seq_len,
                         int advance_seq_len, int64_t max_tokens, void *stream);
/* the same for layers [layer0, layer0+n_layers) in ONE launch (a decode step appends one token to
 * every layer): k_new, v_new [n_layers, batch, n_new, n_kv_heads, d_h]. */
int bgtq_quantize_append_layers(const bgtq_layout *layout, int layer0, int n_layers, void *cache,
                                const void *k_new, const void *v_new, int dt, int batch, int n_new,
                                int32_t *seq_len, int advance_seq_len, int64_t max_tokens, void *stream);

/* ---- a5 + a6: split-KV decode attention over the packed cache with the exact
 * log-sum-exp merge across splits and the V de-rotation.  For every sequence s and
 * query head a:  out = softmax_t(softmax_scale * <q, khat_t>) . vhat_t  over t in [0, seq_len[s]),
 * khat/vhat the dequantised cache (never materialised).  seq_len[s] = 0 gives zeros.
 * q [device] bf16 [n_layers_per_call, batch, n_q_heads, d_h]; out [device] bf16, same shape.
 * bgtq_decode_attention: one layer.  bgtq_decode_attention_layers: layers
 *   [layer0, layer0+n_layers) as independent problems in ONE launch (BASELINE.json cfg2
 *   "36 independent layers").
 * workspace [device] >= bgtq_workspace_bytes(layout, batch, n_layers).
 * Stream semantics: the call enqueues three kernels (query fold, split-KV attention, merge) chained by programmatic
 *   dependent launch; the first of them is itself launched programmatically, so that in a layer-by-layer decode its
 *   prologue runs beside the previous call's merge kernel.  It reads q BEFORE its griddepcontrol.wait: q (like the cache
 *   and seq_len) must come from work that precedes the call on `stream` in the ordinary sense -- a kernel that does not
 *   itself signal griddepcontrol.launch_dependents before it has written q (no kernel of this library writes q).
 *   The workspace may be shared by consecutive calls on one stream; calls on different streams need their own. */
int bgtq_decode_attention(const bgtq_layout *layout, int layer, const void *cache, const void *q,
                          const int32_t *seq_len, int batch, int64_t max_tokens,
                          float softmax_scale, void *out, void *workspace, size_t workspace_bytes,
                          void *stream);
int bgtq_decode_attention_layers(const bgtq_layout *layout, int layer0, int n_layers,
                                 const void *cache, const void *q, const int32_t *seq_len,
                                 int batch, int64_t max_tokens, float softmax_scale, void *out,
                                 void *workspace, size_t workspace_bytes, void *stream);

/* ---- SURVEY.md 8(f).4 "protected windows": decode attention in the paper's *protected-buffer* regime,
 * the cache is [sink (fp16) | compressed | recent (fp16)] -- the first n_sink tokens and
 * the most recent n_recent tokens of every sequence are attended from fp16 rows, every other token from the
 * packed cache; one exact softmax over all seq_len[s] tokens (the three parts are merged by the same
 * log-sum-exp rule as the key-axis splits).  The paper uses n_sink = 4, n_recent = 128.
 * win_k, win_v [device] fp16 [n_layers_of_the_layout, batch, n_kv_heads, n_sink + n_recent, d_h]
 *   (bgtq_window_bytes each): slot j < n_sink holds token j (post-RoPE key / value), slot
 *   n_sink + (t mod n_recent) holds token t >= n_sink while it is among the last n_recent.  The windows of
 *   layers [layer0, layer0 + n_layers) are read.  The packed cache still holds EVERY token (append quantises
 *   as usual); its tokens outside [n_sink, seq_len - n_recent) are skipped / masked, never read as keys.
 * Limits: 0 <= n_sink < 128, n_recent >= 0, 1 <= n_sink + n_recent <= 1024 (else BGTQ_EINVAL; use
 *   bgtq_decode_attention_layers for the buffer-free path).  Everything else as bgtq_decode_attention_layers.
 *   Contiguous cache layout only (no paged variant).
 * bgtq_window_append: fp16 copies (round-to-nearest-even) of the n_new tokens the matching
 *   bgtq_quantize_append_layers call stores at positions seq_len[s] .. seq_len[s] + n_new - 1, written to their
 *   window slots; call it BEFORE that append advances seq_len.  k_new (post-RoPE), v_new, dt, batch, n_new as
 *   there; max_tokens is that append's capacity: tokens at positions >= max_tokens are dropped here exactly as the
 *   append drops them (the ring keeps the rows of the tokens that ARE cached).  The window limits of
 *   bgtq_decode_attention_protected apply (else BGTQ_EINVAL).  Caller owns all buffers. */
size_t bgtq_window_bytes(const bgtq_layout *layout, int batch, int n_sink, int n_recent);
int bgtq_window_append(const bgtq_layout *layout, int layer0, int n_layers, const void *k_new,
                       const void *v_new, int dt, int batch, int n_new, const int32_t *seq_len,
                       int64_t max_tokens, void *win_k, void *win_v, int n_sink, int n_recent, void *stream);
int bgtq_decode_attention_protected(const bgtq_layout *layout, int layer0, int n_layers, const void *cache,
                                    const void *q, const int32_t *seq_len, int batch, int64_t max_tokens,
                                    float softmax_scale, const void *win_k, const void *win_v, int n_sink,
                                    int n_recent, void *out, void *workspace, size_t workspace_bytes,
                                    void *stream);

/* ---- SURVEY.md 8(f).4 "RoPE fused into append": bgtq_quantize_append_layers on PRE-RoPE keys.
 * k_pre [device] [n_layers, batch, n_new, n_kv_heads, d_h] of dtype dt; the token stored at cache position
 * t is first rotated block by block (the layout's pairing):
 *     a' = x_a * cos[t][i] - x_b * sin[t][i],   b' = x_a * sin[t][i] + x_b * cos[t][i]
 * with rope_cos, rope_sin [device] fp32 [rope_rows, d_h/2] (rope_rows >= max_tokens, else
 * BGTQ_ECAPACITY), evaluated in fp64 -- both products are exact, so each output is the correctly
 * rounded value of the expression -- and quantised WITHOUT an intermediate rounding to dt (PAPER.md:122
 * quantises post-RoPE keys; this saves the separate rotary pass and its K write + read).  V and all
 * other arguments as for bgtq_quantize_append_layers. */
int bgtq_quantize_append_rope(const bgtq_layout *layout, int layer0, int n_layers, void *cache,
                              const void *k_pre, const void *v_new, int dt, int batch, int n_new,
                              int32_t *seq_len, int advance_seq_len, int64_t max_tokens,
                              const float *rope_cos, const float *rope_sin, int64_t rope_rows, void *stream);

/* ---- SURVEY.md 8(f).4 "paged sequences": the same two calls over a PAGED cache.
 * The cache is a set of pools, one per (layer, kv head), each of n_pages pages; a page is one
 * 128-token tile of that head (bgtq_tile_stride bytes, the same tile format as the contiguous
 * layout).  Pool (layer, kv_head) starts at byte bgtq_paged_pool_offset(...).
 * page_table [device] int32 [batch, table_stride]: page_table[s][j] = page that holds tokens
 * [128 j, 128 j + 128) of sequence s, the same index in every (layer, head) pool (one logical block
 * id per 128 tokens, as in a paged serving cache).  Entries are read only for tiles below
 * ceil(seq_len[s]/128) (decode) or touched by the new tokens (append); they must be in
 * [0, n_pages) and distinct across live tiles -- not checked on the device.  Capacity per sequence
 * is 128 * table_stride tokens; everything else (arguments, arithmetic, results) is as for the
 * contiguous calls above: a paged cache holds byte-identical tiles, only their addresses differ. */
size_t bgtq_paged_cache_bytes(const bgtq_layout *layout, int64_t n_pages);
int64_t bgtq_paged_pool_offset(const bgtq_layout *layout, int layer, int kv_head, int64_t n_pages);
int bgtq_quantize_append_paged(const bgtq_layout *layout, int layer0, int n_layers, void *cache,
                               const void *k_new, const void *v_new, int dt, int batch, int n_new,
                               int32_t *seq_len, int advance_seq_len, const int32_t *page_table,
                               int table_stride, int64_t n_pages, void *stream);
int bgtq_decode_attention_paged(const bgtq_layout *layout, int layer0, int n_layers, const void *cache,
                                const void *q, const int32_t *seq_len, int batch,
                                const int32_t *page_table, int table_stride, int64_t n_pages,
                                float softmax_scale, void *out, void *workspace,
                                size_t workspace_bytes, void *stream);

/* ---- NEXT #1: causal prefill attention over the packed cache.  The chunk's K, V are
 * already in the cache (bgtq_quantize_append first): query token i of sequence s sits at position
 * seq_len[s] - n_q + i and attends to cached tokens [0, that position] (itself included).
 * q, out [device] bf16 [batch, n_q, n_q_heads, d_h] (post-RoPE q); seq_len [device] int32 [batch] >= n_q.
 * A sequence with seq_len[s] < n_q is a caller error the host cannot see: its output rows are zeros.
 * GQA group must be 1, 2, 4 or 8; BGTQ_FORMAT_V1 layouts only.  Runs on the 5th-generation tensor cores (tcgen05.mma with
 * accumulators in tensor memory, warp-specialised). */
size_t bgtq_prefill_workspace_bytes(const bgtq_layout *layout, int batch, int n_q);
int bgtq_prefill_attention(const bgtq_layout *layout, int layer, const void *cache, const void *q,
                           const int32_t *seq_len, int batch, int n_q, int64_t max_tokens, float softmax_scale,
                           void *out, void *workspace, size_t workspace_bytes, void *stream);

/* ---- comparison path (NOT part of the method): the same split-KV decode attention over a
 * plain fp16 cache, so that the paper's "packed cache vs fp16" claims can be restated on
 * this box without a third-party system.  k_cache, v_cache [device] fp16
 * [n_layers, batch, n_kv_heads, max_tokens, d_h] (max_tokens a multiple of 128); q, out bf16
 * [n_layers, batch, n_q_heads, d_h]; out = softmax(scale * q.K^T) V over tokens [0, seq_len[s]). */
size_t bgtq_fp16_workspace_bytes(int batch, int n_layers, int n_kv_heads);
int bgtq_fp16_decode_attention(int n_layers, int batch, int n_q_heads, int n_kv_heads, int d_h,
                               const void *k_cache, const void *v_cache, const void *q,
                               const int32_t *seq_len, int64_t max_tokens, float softmax_scale,
                               void *out, void *workspace, size_t workspace_bytes, void *stream);

/* ---- test hooks (used by tests/ only; synchronous) */
/* decode one unit (b words per lane, 32 lanes, plane-major as in a tile) with the kernel's own
 * unpack routine: words [host] uint32 [b*32] -> values [host] float [32 lanes][32 slots]. */
int bgtq_debug_decode_unit(int b, const uint32_t *words, float *values);
/* bgtq_quantize_append* with >= 16 new tokens per sequence runs the tensor-core fast paths (TF32 hi/lo products, codes inside
 * a guard band of a threshold recomputed with the exact fp64 chain: same bytes as the exact kernel; whole tiles of new
 * tokens in quantize_tile_kernel, the rest in the sub-batch kernel).  on != 0 forces the exact fp64 sub-batch kernel for
 * every tile of every call of the process (tests compare the two; bench.py times both).  Returns the old setting. */
int bgtq_debug_append_exact_only(int on);
/* measurement hook for bench.py's roofline: while enabled, every decode call records a CUDA event
 * pair on its stream around the split-KV decode kernel alone (not the q-fold / combine kernels);
 * _read synchronises those events, returns the summed milliseconds and the number of launches
 * since the last read, and resets.  Do not enable during stream capture. */
void bgtq_profile_decode(int enable);
int bgtq_profile_decode_read(double *ms_sum, int *count);
/* instruction-rate microbenchmarks behind the numbers DESIGN.md section 7 and profiles/ quote (which pipes the unpack
 * instructions share, what a 3-bit unit costs to unpack, how fast one thread issues tcgen05.mma); `warps` = warps per SM
 * (4..16) for the pipe and unpack tests.  which in [0, BGTQ_MICROBENCH_COUNT); bgtq_debug_microbench_name gives the
 * quantity and its unit.  Synchronous, about 10 ms each; not part of the method. */
#define BGTQ_MICROBENCH_COUNT 22
const char *bgtq_debug_microbench_name(int which);
int bgtq_debug_microbench(int which, int warps, double *value);
/* number of kernels launched by this library since load (bench.py's gpu_launches). */
int64_t bgtq_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* BGTQ_H */
