// bgtq_host.cu -- host side of the C-ABI: argument checks, layout build, host
// allocator (a2), sizes.  No arithmetic of the hot path runs here except Alg. 1's host variant.
#include <atomic>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>

#include <cuda_fp16.h>

#include "bgtq_internal.h"

namespace bgtq {

static thread_local std::string g_err;
static std::atomic<int64_t> g_launches{0};

void set_error(const std::string &msg) { g_err = msg; }
int cuda_fail(cudaError_t e, const char *what)
{
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return BGTQ_ECUDA;
}
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
bool first_use_on_device(int key)
{
    static std::mutex mu;
    static bool seen[64][64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64 || key < 0 || key >= 64) return true;
    std::lock_guard<std::mutex> lock(mu);
    const bool first = !seen[key][dev];
    seen[key][dev] = true;
    return first;
}

}  // namespace bgtq

using namespace bgtq;

#define FAIL(code, msg) do { set_error(msg); return (code); } while (0)
#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

extern "C" const char *bgtq_last_error(void) { return g_err.c_str(); }
extern "C" int64_t bgtq_launch_count(void) { return g_launches.load(); }

extern "C" int bgtq_codebook(int b, float *levels)
{
    if (b < 0 || b > BGTQ_MAX_WIDTH || !levels) FAIL(BGTQ_EINVAL, "bgtq_codebook: b in 0..8, levels != NULL");
    double tmp[256];
    codebook_levels(b, tmp);
    for (int k = 0; k < (1 << b); ++k) levels[k] = (float)tmp[k];
    return BGTQ_OK;
}

// ------------------------------------------------------------------ a2, host variant
// Alg. 1 with a linear arg-max; key = 3/4 * s * 4^-b in fp64 (exact: a power-of-two
// scaling of an fp32 value); ties -> smallest index (Q4); zero scores served last in index order (Q5).
static int allocate_host(const float *scores, int n_heads, int L, int b_min, int b_max, int B,
                         uint8_t *bits)
{
    for (int h = 0; h < n_heads; ++h) {
        const float *s = scores + (size_t)h * L;
        uint8_t *b = bits + (size_t)h * L;
        for (int i = 0; i < L; ++i) {
            if (!(s[i] >= 0.0f) || std::isinf(s[i])) FAIL(BGTQ_EINVAL, "bgtq_allocate: scores must be finite and >= 0");
            b[i] = (uint8_t)b_min;
        }
        for (int extra = B - L * b_min; extra > 0; --extra) {
            int best = -1;
            double bestkey = -1.0;
            for (int i = 0; i < L; ++i) {
                if (b[i] >= b_max) continue;
                double key = 0.75 * std::ldexp((double)s[i], -2 * (int)b[i]);
                if (key > bestkey) { bestkey = key; best = i; }
            }
            if (best < 0) break;
            b[best] += 1;
        }
    }
    return BGTQ_OK;
}

extern "C" int bgtq_allocate(const float *scores, int n_heads, int n_blocks, int b_min, int b_max,
                             int total_bits_B, uint8_t *bits, int on_device, void *stream)
{
    if (!scores || !bits || n_heads < 0 || n_blocks <= 0) FAIL(BGTQ_EINVAL, "bgtq_allocate: null pointer or bad shape");
    if (b_min < 0 || b_max > BGTQ_MAX_WIDTH || b_min > b_max) FAIL(BGTQ_EINVAL, "bgtq_allocate: need 0 <= b_min <= b_max <= 8");
    if (total_bits_B < n_blocks * b_min || total_bits_B > n_blocks * b_max)
        FAIL(BGTQ_EBUDGET, "bgtq_allocate: B outside [L*b_min, L*b_max]");
    if (n_heads == 0) return BGTQ_OK;
    if (!on_device) return allocate_host(scores, n_heads, n_blocks, b_min, b_max, total_bits_B, bits);
    if (n_blocks > 1024) FAIL(BGTQ_EINVAL, "bgtq_allocate: device path supports n_blocks <= 1024");
    return launch_allocate(scores, n_heads, n_blocks, b_min, b_max, total_bits_B, bits, (cudaStream_t)stream);
}

// ------------------------------------------------------------------ a1 wrapper
extern "C" size_t bgtq_block_energy_workspace_bytes(int n_q_heads, int n_kv_heads, int d_h)
{
    if (n_q_heads <= 0 || n_kv_heads <= 0 || d_h <= 0) return 0;
    return block_energy_ws_bytes(n_q_heads, n_kv_heads, d_h);
}

extern "C" int bgtq_block_energy(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt,
                                 int n_q_heads, int n_kv_heads, int d_h, int pairing, int kind,
                                 float *scores, float *eq_out, float *ek_out, void *workspace,
                                 size_t workspace_bytes, void *stream)
{
    if (!scores || !workspace) FAIL(BGTQ_EINVAL, "bgtq_block_energy: null scores/workspace");
    if (n_q < 0 || n_k < 0 || (n_q > 0 && !q) || (n_k > 0 && !k)) FAIL(BGTQ_EINVAL, "bgtq_block_energy: bad q/k");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_block_energy: dtype");
    if (n_kv_heads <= 0 || n_q_heads <= 0 || n_q_heads % n_kv_heads) FAIL(BGTQ_EINVAL, "bgtq_block_energy: heads");
    if (d_h <= 0 || d_h % 8 || d_h > 1024) FAIL(BGTQ_EINVAL, "bgtq_block_energy: d_h must be a multiple of 8, <= 1024");
    if (pairing != BGTQ_PAIR_HALF && pairing != BGTQ_PAIR_INTERLEAVED) FAIL(BGTQ_EINVAL, "bgtq_block_energy: pairing");
    if (kind < 0 || kind > BGTQ_Q_ONLY) FAIL(BGTQ_EINVAL, "bgtq_block_energy: score kind");
    if (workspace_bytes < block_energy_ws_bytes(n_q_heads, n_kv_heads, d_h)) FAIL(BGTQ_EWORKSPACE, "bgtq_block_energy: workspace too small");
    return launch_block_energy(q, n_q, k, n_k, dt, n_q_heads, n_kv_heads, d_h, pairing, kind, scores,
                               eq_out, ek_out, workspace, workspace_bytes, (cudaStream_t)stream);
}

static std::atomic<bool> g_append_exact_only{false};
namespace bgtq {
bool append_exact_only() { return g_append_exact_only.load(); }
void set_append_exact_only(bool on) { g_append_exact_only.store(on); }
}  // namespace bgtq
extern "C" int bgtq_debug_append_exact_only(int on) { return g_append_exact_only.exchange(on != 0) ? 1 : 0; }

extern "C" int bgtq_block_energy_static_max_row_elems(void) { return block_energy_static_max_row_elems(); }

extern "C" int bgtq_block_energy_static(const void *q, int64_t n_q, const void *k, int64_t n_k, int dt,
                                        int n_q_heads, int n_kv_heads, int d_h, int pairing, int kind,
                                        float *scores, float *eq_out, float *ek_out, void *stream)
{
    if (!scores) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: null scores");
    if (n_q < 0 || n_k < 0 || (n_q > 0 && !q) || (n_k > 0 && !k)) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: bad q/k");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: dtype");
    if (n_kv_heads <= 0 || n_q_heads <= 0 || n_q_heads % n_kv_heads) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: heads");
    if (d_h <= 0 || d_h % 8 || d_h > 1024) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: d_h must be a multiple of 8, <= 1024");
    if (pairing != BGTQ_PAIR_HALF && pairing != BGTQ_PAIR_INTERLEAVED) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: pairing");
    if (kind < 0 || kind > BGTQ_Q_ONLY) FAIL(BGTQ_EINVAL, "bgtq_block_energy_static: score kind");
    return launch_block_energy_static(q, n_q, k, n_k, dt, n_q_heads, n_kv_heads, d_h, pairing, kind, scores, eq_out, ek_out,
                                      (cudaStream_t)stream);
}

extern "C" size_t bgtq_v_block_energy_workspace_bytes(int n_kv_heads, int d_h)
{
    if (n_kv_heads <= 0 || d_h <= 0) return 0;
    return block_energy_ws_bytes(0, n_kv_heads, d_h);
}

extern "C" int bgtq_v_block_energy(const void *v, int64_t n, int dt, int n_kv_heads, int d_h, float *scores,
                                   void *workspace, size_t workspace_bytes, void *stream)
{
    if (!scores || !workspace) FAIL(BGTQ_EINVAL, "bgtq_v_block_energy: null scores/workspace");
    if (n <= 0 || !v) FAIL(BGTQ_EINVAL, "bgtq_v_block_energy: bad v/n");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_v_block_energy: dtype");
    if (n_kv_heads <= 0) FAIL(BGTQ_EINVAL, "bgtq_v_block_energy: heads");
    if (d_h <= 0 || d_h % BGTQ_V_BLOCK || d_h > 1024) FAIL(BGTQ_EINVAL, "bgtq_v_block_energy: d_h must be a multiple of 16, <= 1024");
    if (workspace_bytes < block_energy_ws_bytes(0, n_kv_heads, d_h)) FAIL(BGTQ_EWORKSPACE, "bgtq_v_block_energy: workspace too small");
    return launch_v_block_energy(v, n, dt, n_kv_heads, d_h, scores, workspace, (cudaStream_t)stream);
}

// ------------------------------------------------------------------ a3: layout build
// Grouping, tile geometry and the k-step program of DESIGN.md section 4.
// V side (reading Q19): same-width groups of 16-coordinate V blocks, ascending width, member blocks ascending; one fp16
// norm row per group, then the groups' code sections (two units of 128 * w bytes per block).  bits_v: 8 widths in 1..8.
// Needs m.vnorm_off; sets everything after it.  All widths equal = the uniform layout of PAPER.md:27, byte for byte.
static void build_v_side(const uint8_t *bits_v, HeadMeta &m)
{
    int nvg = 0, jg = 0;
    for (int w = 1; w <= BGTQ_MAX_WIDTH; ++w) {
        int cnt = 0;
        for (int j = 0; j < kMaxGroups; ++j)
            if (bits_v[j] == w) {
                if (!cnt) { m.vgb[nvg] = (uint8_t)w; m.vgstart[nvg] = (uint8_t)jg; }
                m.vblk[jg] = (uint8_t)j; m.vbg[jg] = (uint8_t)nvg; m.vbw[jg] = (uint8_t)w;
                ++cnt; ++jg;
            }
        if (cnt) m.vgcnt[nvg++] = (uint8_t)cnt;
    }
    m.n_vgroups = (uint8_t)nvg;
    m.b_v = m.vgb[0];
    m.vcode_off = m.vnorm_off + 256 * nvg;
    int off = m.vcode_off;
    for (int j = 0; j < kMaxGroups; ++j) { m.vboff[j] = (uint16_t)off; off += 2 * 128 * m.vbw[j]; }
    m.tile_stride = off;
}

static void build_head_meta(const uint8_t *bits, int d_h, int b_v, const uint8_t *bits_v, int pairing, HeadMeta &m)
{
    std::memset(&m, 0, sizeof(m));
    const int L = d_h / 2;
    m.b_v = b_v;
    int ng = 0, kdim = 0, off = 0, nks = 0;
    for (int w = 1; w <= BGTQ_MAX_WIDTH; ++w) {
        int cnt = 0;
        for (int i = 0; i < L; ++i)
            if (bits[i] == w) {
                int a = pairing == BGTQ_PAIR_HALF ? i : 2 * i;
                int b = pairing == BGTQ_PAIR_HALF ? i + L : 2 * i + 1;
                m.coords[kdim + cnt++] = (uint8_t)a;
                m.coords[kdim + cnt++] = (uint8_t)b;
            }
        if (!cnt) continue;
        m.gb[ng] = (uint8_t)w;
        m.gm[ng] = (uint16_t)cnt;
        m.gstart[ng] = (uint16_t)kdim;
        m.goff[ng] = off;
        // half-steps of 8 coordinates; full one = 128*w bytes, trailing partial (r coords) = 16*r*w
        int n_half = (cnt + 7) / 8;
        for (int j = 0; j < n_half; j += 2) {
            KStep &ks = m.ksteps[nks++];
            int r0 = cnt - 8 * j >= 8 ? 8 : cnt - 8 * j;
            ks.off0 = (uint16_t)(off + j * 128 * w);
            ks.nc0 = (uint8_t)(r0 / 2);
            if (j + 1 < n_half) {
                int r1 = cnt - 8 * (j + 1) >= 8 ? 8 : cnt - 8 * (j + 1);
                ks.off1 = (uint16_t)(off + (j + 1) * 128 * w);
                ks.nc1 = (uint8_t)(r1 / 2);
            } else {
                ks.off1 = 0xFFFF;
                ks.nc1 = 0;
            }
            ks.b = (uint8_t)w;
            ks.flags = (uint8_t)((j == 0 ? 1 : 0) | (j + 2 >= n_half ? 2 : 0) | (ng << 4));
        }
        off += 16 * cnt * w;
        kdim += cnt;
        ++ng;
    }
    m.n_groups = ng;
    m.kdim = kdim;
    m.n_ksteps = nks;
    m.kcode_bytes = off;
    m.knorm_off = off;
    m.vnorm_off = off + 256 * ng;
    uint8_t uni[kMaxGroups];
    for (int j = 0; j < kMaxGroups; ++j) uni[j] = (uint8_t)b_v;
    build_v_side(bits_v ? bits_v : uni, m);
}

// BGTQ-v2: words per lane of a chunk of r slots at width b
static int chunk_words(int b, int r)
{
    const int nwm = r > 24 ? 3 : (r + 7) / 8;
    switch (b) {
    case 1: return 1;
    case 2: return (r + 15) / 16;
    case 3: return nwm;
    case 4: return nwm + 1;
    default: return (r * b + 31) / 32;
    }
}

static void build_head_meta_v2(const uint8_t *bits, int d_h, int b_v, int pairing, HeadMeta &m)
{
    std::memset(&m, 0, sizeof(m));
    const int L = d_h / 2;
    m.b_v = b_v;
    m.format = 2;
    int ng = 0, kdim = 0, off = 0, nch = 0;
    for (int w = 1; w <= BGTQ_MAX_WIDTH; ++w) {
        int cnt = 0;
        for (int i = 0; i < L; ++i)
            if (bits[i] == w) {
                int a = pairing == BGTQ_PAIR_HALF ? i : 2 * i;
                int b = pairing == BGTQ_PAIR_HALF ? i + L : 2 * i + 1;
                m.coords[kdim + cnt++] = (uint8_t)a;
                m.coords[kdim + cnt++] = (uint8_t)b;
            }
        if (!cnt) continue;
        m.gb[ng] = (uint8_t)w;
        m.gm[ng] = (uint16_t)cnt;
        m.gstart[ng] = (uint16_t)kdim;
        m.goff[ng] = off;
        for (int u = 0; 32 * u < cnt; ++u) {
            Chunk2 &c = m.chunks[nch++];
            const int r = cnt - 32 * u >= 32 ? 32 : cnt - 32 * u;
            c.off = (uint16_t)off;
            c.ustart = (uint16_t)(kdim + 32 * u);
            c.b = (uint8_t)w;
            c.r = (uint8_t)r;
            c.nw = (uint8_t)chunk_words(w, r);
            c.flags = (uint8_t)((u == 0 ? 1 : 0) | (ng << 4));
            off += 128 * c.nw;
        }
        kdim += cnt;
        ++ng;
    }
    m.n_groups = ng;
    m.kdim = kdim;
    m.n_ksteps = nch;
    m.kcode_bytes = 4 * off;                 // four quadrants of 32 tokens
    m.knorm_off = m.kcode_bytes;
    m.vnorm_off = m.knorm_off + 256 * ng;
    m.vcode_off = m.vnorm_off + 256;
    m.tile_stride = m.vcode_off + 16 * d_h * b_v;
    m.n_vgroups = 1;                         // (row order keeps one V group: bits_v is a BGTQ-v1 feature)
    m.vgb[0] = (uint8_t)b_v; m.vgcnt[0] = kMaxGroups;
    for (int j = 0; j < kMaxGroups; ++j) { m.vblk[j] = (uint8_t)j; m.vbw[j] = (uint8_t)b_v; }
}

extern "C" int bgtq_layout_create(const uint8_t *bits, int n_layers, int n_kv_heads, int n_q_heads,
                                  int d_h, int b_v, int pairing, const float *rotations,
                                  bgtq_layout **out)
{
    return bgtq_layout_create_format(bits, n_layers, n_kv_heads, n_q_heads, d_h, b_v, pairing, rotations,
                                     BGTQ_FORMAT_V1, out);
}

extern "C" int bgtq_layout_format(const bgtq_layout *lay) { return lay ? (lay->format | (lay->cb_exact ? BGTQ_CODEBOOK_EXACT : 0)) : 0; }

extern "C" int bgtq_codebook_exact(int b, int m, float *levels)
{
    if (b < 0 || b > BGTQ_MAX_WIDTH || m < 2 || m > 1024 || (m & 1) || !levels)
        FAIL(BGTQ_EINVAL, "bgtq_codebook_exact: b in 0..8, m even in 2..1024, levels != NULL");
    double tmp[256];
    codebook_levels_sphere(b, m, tmp);
    for (int k = 0; k < (1 << b); ++k) levels[k] = (float)tmp[k];
    return BGTQ_OK;
}

static int layout_create_impl(const uint8_t *bits, const uint8_t *bits_v, int n_layers, int n_kv_heads, int n_q_heads,
                              int d_h, int b_v, int pairing, const float *rotations, int format, bgtq_layout **out);

extern "C" int bgtq_layout_create_format(const uint8_t *bits, int n_layers, int n_kv_heads, int n_q_heads,
                                         int d_h, int b_v, int pairing, const float *rotations, int format,
                                         bgtq_layout **out)
{
    if (b_v < 1 || b_v > BGTQ_MAX_WIDTH) FAIL(BGTQ_EINVAL, "bgtq_layout_create: b_v in 1..8");
    return layout_create_impl(bits, nullptr, n_layers, n_kv_heads, n_q_heads, d_h, b_v, pairing, rotations, format, out);
}

extern "C" int bgtq_layout_create_kv(const uint8_t *bits_k, const uint8_t *bits_v, int n_layers, int n_kv_heads,
                                     int n_q_heads, int d_h, int pairing, const float *rotations, int format,
                                     bgtq_layout **out)
{
    if (!bits_v) FAIL(BGTQ_EINVAL, "bgtq_layout_create_kv: null pointer");
    if (d_h != kDh) FAIL(BGTQ_EINVAL, "bgtq_layout_create_kv: d_h must be 128");
    if ((format & ~BGTQ_CODEBOOK_EXACT) != BGTQ_FORMAT_V1) FAIL(BGTQ_EINVAL, "bgtq_layout_create_kv: V-side widths are built for BGTQ_FORMAT_V1 layouts");
    if (n_layers > 0 && n_kv_heads > 0)
        for (size_t i = 0; i < (size_t)n_layers * n_kv_heads * (d_h / BGTQ_V_BLOCK); ++i)
            if (bits_v[i] < 1 || bits_v[i] > BGTQ_MAX_WIDTH) FAIL(BGTQ_EINVAL, "bgtq_layout_create_kv: V widths must be 1..8");
    return layout_create_impl(bits_k, bits_v, n_layers, n_kv_heads, n_q_heads, d_h, 0, pairing, rotations, format, out);
}

static int layout_create_impl(const uint8_t *bits, const uint8_t *bits_v, int n_layers, int n_kv_heads, int n_q_heads,
                              int d_h, int b_v, int pairing, const float *rotations, int format, bgtq_layout **out)
{
    if (!bits || !rotations || !out) FAIL(BGTQ_EINVAL, "bgtq_layout_create: null pointer");
    const int cb_exact = (format & BGTQ_CODEBOOK_EXACT) ? 1 : 0;
    format &= ~BGTQ_CODEBOOK_EXACT;
    if (format != BGTQ_FORMAT_V1 && format != BGTQ_FORMAT_V2) FAIL(BGTQ_EINVAL, "bgtq_layout_create: format must be BGTQ_FORMAT_V1 or BGTQ_FORMAT_V2");
    if (cb_exact && format != BGTQ_FORMAT_V1) FAIL(BGTQ_EINVAL, "bgtq_layout_create: BGTQ_CODEBOOK_EXACT is built for BGTQ_FORMAT_V1 layouts");
    if (d_h != kDh) FAIL(BGTQ_EINVAL, "bgtq_layout_create: d_h must be 128");
    if (n_layers <= 0 || n_kv_heads <= 0 || n_q_heads <= 0 || n_q_heads % n_kv_heads)
        FAIL(BGTQ_EINVAL, "bgtq_layout_create: bad layer/head counts");
    if (n_q_heads / n_kv_heads > 8) FAIL(BGTQ_EINVAL, "bgtq_layout_create: GQA group size must be <= 8");
    if (pairing != BGTQ_PAIR_HALF && pairing != BGTQ_PAIR_INTERLEAVED) FAIL(BGTQ_EINVAL, "bgtq_layout_create: pairing");
    const int L = d_h / 2;
    for (size_t i = 0; i < (size_t)n_layers * n_kv_heads * L; ++i)
        if (bits[i] > BGTQ_MAX_WIDTH) FAIL(BGTQ_EINVAL, "bgtq_layout_create: widths must be 0..8");

    bgtq_layout *lay = new (std::nothrow) bgtq_layout();
    if (!lay) FAIL(BGTQ_EINVAL, "bgtq_layout_create: out of host memory");
    lay->n_layers = n_layers; lay->n_kv_heads = n_kv_heads; lay->n_q_heads = n_q_heads;
    lay->d_h = d_h; lay->b_v = b_v; lay->pairing = pairing;
    lay->format = format; lay->d_planes = nullptr;
    lay->cb_exact = cb_exact; lay->d_hcb16 = nullptr; lay->d_hcb64 = nullptr;
    lay->d_meta = nullptr; lay->d_rot = nullptr; lay->d_rot_t = nullptr; lay->d_rot_hl = nullptr; lay->d_cb16 = nullptr; lay->d_cb64 = nullptr;
    lay->meta.resize((size_t)n_layers * n_kv_heads);
    int64_t prefix = 0;
    lay->max_stride = 0;
    lay->max_chunks = 0;
    lay->v_grouped = 0;
    lay->max_rows = 1;
    for (int l = 0; l < n_layers; ++l) {
        int64_t lsum = 0;
        for (int h = 0; h < n_kv_heads; ++h) {
            HeadMeta &m = lay->meta[(size_t)l * n_kv_heads + h];
            if (format == BGTQ_FORMAT_V2) build_head_meta_v2(bits + ((size_t)l * n_kv_heads + h) * L, d_h, b_v, pairing, m);
            else build_head_meta(bits + ((size_t)l * n_kv_heads + h) * L, d_h, b_v,
                                 bits_v ? bits_v + ((size_t)l * n_kv_heads + h) * kMaxGroups : nullptr, pairing, m);
            m.format = format;
            if (m.n_vgroups > 1) lay->v_grouped = 1;
            if (m.n_groups + m.n_vgroups > lay->max_rows) lay->max_rows = m.n_groups + m.n_vgroups;
            m.layer_prefix = prefix;
            m.head_prefix = lsum;
            lsum += m.tile_stride;
            if (m.tile_stride > lay->max_stride) lay->max_stride = m.tile_stride;
            if (format == BGTQ_FORMAT_V2 && m.n_ksteps > lay->max_chunks) lay->max_chunks = m.n_ksteps;
        }
        for (int h = 0; h < n_kv_heads; ++h) lay->meta[(size_t)l * n_kv_heads + h].layer_sum = lsum;
        prefix += lsum;
    }
    lay->total_stride_sum = prefix;

    // device copies: metadata, rotation table (both orientations), codebooks
    const int64_t rot_n = rot_offset(d_h + 2);
    std::vector<float> rot_t((size_t)rot_n);
    for (int m = 2; m <= d_h; m += 2) {
        const float *P = rotations + rot_offset(m);
        float *T = rot_t.data() + rot_offset(m);
        for (int j = 0; j < m; ++j)
            for (int k = 0; k < m; ++k) T[(size_t)k * m + j] = P[(size_t)j * m + k];
    }
    std::vector<float2> rot_hl((size_t)rot_n);        // hi = Pi rounded to TF32 (10-bit mantissa, ties away), lo = Pi - hi (exact)
    for (int64_t i = 0; i < rot_n; ++i) {
        uint32_t u;
        std::memcpy(&u, &rotations[i], 4);
        u = (u + 0x1000u) & 0xFFFFE000u;
        float hi;
        std::memcpy(&hi, &u, 4);
        rot_hl[(size_t)i] = make_float2(hi, rotations[i] - hi);
    }
    std::vector<uint16_t> cb16(512, 0);
    std::vector<double> cb64(512, 0.0);
    for (int b = 0; b <= BGTQ_MAX_WIDTH; ++b) {
        double lv[256];
        codebook_levels(b, lv);
        for (int k = 0; k < (1 << b); ++k) {
            cb64[(1 << b) - 1 + k] = lv[k];
            __half hv = __double2half(lv[k]);
            uint16_t u;
            std::memcpy(&u, &hv, 2);
            cb16[(1 << b) - 1 + k] = u;
        }
    }
    // exact-density tables per (layer, kv head): flat by width like the shared table; widths without a group keep the
    // Gaussian levels (never used)
    std::vector<uint16_t> hcb16;
    std::vector<double> hcb64;
    if (cb_exact) {
        const size_t nh = lay->meta.size();
        hcb16.assign(nh * 2 * kHeadLutHalves, 0);
        hcb64.assign(nh * 2 * 512, 0.0);
        std::vector<std::vector<double>> cache_lv(9 * 65);         // (b, m/2) -> levels, solved once
        auto levels_of = [&](int b, int m) -> const std::vector<double> & {
            std::vector<double> &v = cache_lv[(size_t)b * 65 + m / 2];
            if (v.empty()) { v.resize(1 << b); codebook_levels_sphere(b, m, v.data()); }
            return v;
        };
        for (size_t hi = 0; hi < nh; ++hi) {
            const HeadMeta &m = lay->meta[hi];
            for (int side = 0; side < 2; ++side) {
                uint16_t *t16 = hcb16.data() + (hi * 2 + side) * kHeadLutHalves;
                double *t64 = hcb64.data() + (hi * 2 + side) * 512;
                for (int i = 0; i < 512; ++i) { t16[i] = cb16[i < 511 ? i : 510]; t64[i] = cb64[i < 511 ? i : 510]; }
                auto put = [&](int b, int mm) {
                    const std::vector<double> &lv = levels_of(b, mm);
                    for (int k = 0; k < (1 << b); ++k) {
                        t64[(1 << b) - 1 + k] = lv[k];
                        __half hv = __double2half(lv[k]);
                        std::memcpy(&t16[(1 << b) - 1 + k], &hv, 2);
                    }
                };
                if (side == 0) for (int g = 0; g < m.n_groups; ++g) put(m.gb[g], m.gm[g]);
                else for (int g = 0; g < m.n_vgroups; ++g) put(m.vgb[g], 16 * m.vgcnt[g]);
                uint32_t *pair = reinterpret_cast<uint32_t *>(t16 + 512);     // two adjacent 5-bit codes -> fp16x2
                for (int i = 0; i < 1024; ++i) pair[i] = (uint32_t)t16[31 + (i & 31)] | ((uint32_t)t16[31 + (i >> 5)] << 16);
            }
        }
    }
    std::vector<uint8_t> planes(kPlaneBytes, 0);
    lay->kappa[0] = 1.f;
    for (int b = 1; b <= BGTQ_MAX_WIDTH; ++b)
        codebook_planes(b, &lay->kappa[b], planes.data() + (1 << b) - 1, planes.data() + 512 + (1 << b) - 1);
    cudaError_t e = cudaSuccess;
    int dev = 0;
    if (e == cudaSuccess) e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&lay->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_meta, lay->meta.size() * sizeof(HeadMeta));
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_rot, rot_n * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_rot_t, rot_n * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_rot_hl, rot_n * sizeof(float2));
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_rot_hl, rot_hl.data(), rot_n * sizeof(float2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_cb16, 512 * sizeof(uint16_t));
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_cb64, 512 * sizeof(double));
    if (e == cudaSuccess && cb_exact) e = cudaMalloc(&lay->d_hcb16, hcb16.size() * sizeof(uint16_t));
    if (e == cudaSuccess && cb_exact) e = cudaMalloc(&lay->d_hcb64, hcb64.size() * sizeof(double));
    if (e == cudaSuccess && cb_exact) e = cudaMemcpy(lay->d_hcb16, hcb16.data(), hcb16.size() * sizeof(uint16_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && cb_exact) e = cudaMemcpy(lay->d_hcb64, hcb64.data(), hcb64.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&lay->d_planes, kPlaneBytes);
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_planes, planes.data(), kPlaneBytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_meta, lay->meta.data(), lay->meta.size() * sizeof(HeadMeta), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_rot, rotations, rot_n * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_rot_t, rot_t.data(), rot_n * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_cb16, cb16.data(), 512 * sizeof(uint16_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(lay->d_cb64, cb64.data(), 512 * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        bgtq_layout_destroy(lay);
        return cuda_fail(e, "bgtq_layout_create");
    }
    *out = lay;
    return BGTQ_OK;
}

extern "C" void bgtq_layout_destroy(bgtq_layout *lay)
{
    if (!lay) return;
    cudaFree(lay->d_meta); cudaFree(lay->d_rot); cudaFree(lay->d_rot_t); cudaFree(lay->d_rot_hl);
    cudaFree(lay->d_cb16); cudaFree(lay->d_cb64); cudaFree(lay->d_planes); cudaFree(lay->d_hcb16); cudaFree(lay->d_hcb64);
    delete lay;
}

static inline int64_t n_cap_tiles(int64_t max_tokens) { return (max_tokens + kTile - 1) / kTile; }

extern "C" size_t bgtq_cache_bytes(const bgtq_layout *lay, int batch, int64_t max_tokens)
{
    if (!lay || batch <= 0 || max_tokens <= 0) return 0;
    return (size_t)(n_cap_tiles(max_tokens) * batch * lay->total_stride_sum);
}
extern "C" double bgtq_token_bytes(const bgtq_layout *lay, int layer, int kv_head)
{
    if (!lay || layer < 0 || layer >= lay->n_layers || kv_head < 0 || kv_head >= lay->n_kv_heads) return 0.0;
    return lay->meta[(size_t)layer * lay->n_kv_heads + kv_head].tile_stride / (double)kTile;
}
extern "C" int64_t bgtq_tile_stride(const bgtq_layout *lay, int layer, int kv_head)
{
    if (!lay || layer < 0 || layer >= lay->n_layers || kv_head < 0 || kv_head >= lay->n_kv_heads) return -1;
    return lay->meta[(size_t)layer * lay->n_kv_heads + kv_head].tile_stride;
}
extern "C" int64_t bgtq_region_offset(const bgtq_layout *lay, int layer, int seq, int kv_head,
                                      int batch, int64_t max_tokens)
{
    if (!lay || layer < 0 || layer >= lay->n_layers || kv_head < 0 || kv_head >= lay->n_kv_heads ||
        seq < 0 || seq >= batch || max_tokens <= 0) return -1;
    const HeadMeta &m = lay->meta[(size_t)layer * lay->n_kv_heads + kv_head];
    return n_cap_tiles(max_tokens) * ((int64_t)batch * m.layer_prefix + (int64_t)seq * m.layer_sum + m.head_prefix);
}
static size_t decode_ws_any(const bgtq_layout *lay, int batch, int n_layers);
extern "C" size_t bgtq_workspace_bytes(const bgtq_layout *lay, int batch, int n_layers_per_call)
{
    if (!lay || batch <= 0 || n_layers_per_call <= 0) return 0;
    return decode_ws_any(lay, batch, n_layers_per_call);
}

// split-KV decode: the BGTQ-v1 mma.sync kernel or the BGTQ-v2 tcgen05 kernel, by the layout's format
static size_t decode_ws_any(const bgtq_layout *lay, int batch, int n_layers)
{
    return lay->format == 2 ? decode2_ws_bytes(lay, batch, n_layers) : decode_ws_bytes(lay, batch, n_layers);
}
static int launch_decode_any(const bgtq_layout *lay, int layer0, int n_layers, const void *cache, const void *q,
                             const int32_t *seq_len, int batch, int64_t max_tokens, float scale, void *out, void *ws,
                             size_t ws_bytes, const PageMap *pm, cudaStream_t st, const Window *win = nullptr)
{
    if (lay->format == 2) return launch_decode2(lay, layer0, n_layers, cache, q, seq_len, batch, max_tokens, scale, out, ws, ws_bytes, pm, st, win);
    return launch_decode(lay, layer0, n_layers, cache, q, seq_len, batch, max_tokens, scale, out, ws, ws_bytes, pm, st, win);
}

// ------------------------------------------------------------------ a4 / a5 wrappers
extern "C" int bgtq_quantize_append_layers(const bgtq_layout *lay, int layer0, int n_layers, void *cache,
                                           const void *k_new, const void *v_new, int dt, int batch, int n_new,
                                           int32_t *seq_len, int advance_seq_len, int64_t max_tokens, void *stream)
{
    if (!lay || !cache || !seq_len) FAIL(BGTQ_EINVAL, "bgtq_quantize_append: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_quantize_append: layer out of range");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_quantize_append: dtype");
    if (batch <= 0 || n_new < 0 || max_tokens <= 0) FAIL(BGTQ_EINVAL, "bgtq_quantize_append: batch/n_new/max_tokens");
    if (batch > 65535 || (int64_t)n_layers * lay->n_kv_heads > 65535) FAIL(BGTQ_EINVAL, "bgtq_quantize_append: batch or layers*heads > 65535");
    if (n_new > max_tokens) FAIL(BGTQ_ECAPACITY, "bgtq_quantize_append: n_new exceeds max_tokens");
    if (n_new == 0) return BGTQ_OK;
    if (!k_new || !v_new) FAIL(BGTQ_EINVAL, "bgtq_quantize_append: null k_new/v_new");
    return launch_quantize_append(lay, layer0, n_layers, cache, k_new, v_new, dt, batch, n_new, seq_len,
                                  advance_seq_len, max_tokens, nullptr, nullptr, (cudaStream_t)stream);
}

// ------------------------------------------------------------------ RoPE fused into append
extern "C" int bgtq_quantize_append_rope(const bgtq_layout *lay, int layer0, int n_layers, void *cache,
                                         const void *k_pre, const void *v_new, int dt, int batch, int n_new,
                                         int32_t *seq_len, int advance_seq_len, int64_t max_tokens,
                                         const float *rope_cos, const float *rope_sin, int64_t rope_rows, void *stream)
{
    if (!lay || !cache || !seq_len || !rope_cos || !rope_sin) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_rope: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_rope: layer out of range");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_rope: dtype");
    if (batch <= 0 || n_new < 0 || max_tokens <= 0) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_rope: batch/n_new/max_tokens");
    if (batch > 65535 || (int64_t)n_layers * lay->n_kv_heads > 65535) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_rope: batch or layers*heads > 65535");
    if (n_new > max_tokens) FAIL(BGTQ_ECAPACITY, "bgtq_quantize_append_rope: n_new exceeds max_tokens");
    if (rope_rows < max_tokens) FAIL(BGTQ_ECAPACITY, "bgtq_quantize_append_rope: cos/sin tables have fewer rows than max_tokens");
    if (n_new == 0) return BGTQ_OK;
    if (!k_pre || !v_new) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_rope: null k_pre/v_new");
    const RopeTab rt{rope_cos, rope_sin};
    return launch_quantize_append(lay, layer0, n_layers, cache, k_pre, v_new, dt, batch, n_new, seq_len,
                                  advance_seq_len, max_tokens, nullptr, &rt, (cudaStream_t)stream);
}

// ------------------------------------------------------------------ paged cache
extern "C" size_t bgtq_paged_cache_bytes(const bgtq_layout *lay, int64_t n_pages)
{
    if (!lay || n_pages <= 0) return 0;
    return (size_t)(n_pages * lay->total_stride_sum);
}
extern "C" int64_t bgtq_paged_pool_offset(const bgtq_layout *lay, int layer, int kv_head, int64_t n_pages)
{
    if (!lay || layer < 0 || layer >= lay->n_layers || kv_head < 0 || kv_head >= lay->n_kv_heads || n_pages <= 0) return -1;
    const HeadMeta &m = lay->meta[(size_t)layer * lay->n_kv_heads + kv_head];
    return n_pages * ((int64_t)m.layer_prefix + m.head_prefix);
}
extern "C" int bgtq_quantize_append_paged(const bgtq_layout *lay, int layer0, int n_layers, void *cache,
                                          const void *k_new, const void *v_new, int dt, int batch, int n_new,
                                          int32_t *seq_len, int advance_seq_len, const int32_t *page_table,
                                          int table_stride, int64_t n_pages, void *stream)
{
    if (!lay || !cache || !seq_len || !page_table) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_paged: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_paged: layer out of range");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_paged: dtype");
    if (batch <= 0 || n_new < 0 || table_stride <= 0 || n_pages <= 0) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_paged: batch/n_new/table_stride/n_pages");
    if (batch > 65535 || (int64_t)n_layers * lay->n_kv_heads > 65535) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_paged: batch or layers*heads > 65535");
    const int64_t max_tokens = (int64_t)table_stride * kTile;
    if (n_new > max_tokens) FAIL(BGTQ_ECAPACITY, "bgtq_quantize_append_paged: n_new exceeds 128 * table_stride");
    if (n_new == 0) return BGTQ_OK;
    if (!k_new || !v_new) FAIL(BGTQ_EINVAL, "bgtq_quantize_append_paged: null k_new/v_new");
    const PageMap pm{page_table, table_stride, n_pages};
    return launch_quantize_append(lay, layer0, n_layers, cache, k_new, v_new, dt, batch, n_new, seq_len,
                                  advance_seq_len, max_tokens, &pm, nullptr, (cudaStream_t)stream);
}
extern "C" int bgtq_decode_attention_paged(const bgtq_layout *lay, int layer0, int n_layers, const void *cache,
                                           const void *q, const int32_t *seq_len, int batch,
                                           const int32_t *page_table, int table_stride, int64_t n_pages,
                                           float softmax_scale, void *out, void *workspace,
                                           size_t workspace_bytes, void *stream)
{
    if (!lay || !cache || !q || !seq_len || !out || !workspace || !page_table) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_paged: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_paged: layer range");
    if (batch <= 0 || table_stride <= 0 || n_pages <= 0) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_paged: batch/table_stride/n_pages");
    if (!(softmax_scale > 0.0f) || std::isinf(softmax_scale)) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_paged: softmax_scale must be finite and > 0");
    if (lay->cb_exact || lay->v_grouped) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_paged: not built for BGTQ_CODEBOOK_EXACT layouts or V-side groups");
    if (workspace_bytes < decode_ws_any(lay, batch, n_layers)) FAIL(BGTQ_EWORKSPACE, "bgtq_decode_attention_paged: workspace too small");
    const PageMap pm{page_table, table_stride, n_pages};
    return launch_decode_any(lay, layer0, n_layers, cache, q, seq_len, batch, (int64_t)table_stride * kTile, softmax_scale,
                             out, workspace, workspace_bytes, &pm, (cudaStream_t)stream);
}

extern "C" int bgtq_quantize_append(const bgtq_layout *lay, int layer, void *cache, const void *k_new,
                                    const void *v_new, int dt, int batch, int n_new, int32_t *seq_len,
                                    int advance_seq_len, int64_t max_tokens, void *stream)
{
    return bgtq_quantize_append_layers(lay, layer, 1, cache, k_new, v_new, dt, batch, n_new, seq_len,
                                       advance_seq_len, max_tokens, stream);
}

extern "C" const char *bgtq_debug_microbench_name(int which) { return microbench_name(which); }
extern "C" int bgtq_debug_microbench(int which, int warps, double *value)
{
    if (!value || warps < 1 || warps > 16) FAIL(BGTQ_EINVAL, "bgtq_debug_microbench: value != NULL, warps in 1..16");
    return microbench_run(which, warps, value);
}
extern "C" void bgtq_profile_decode(int enable) { profile_decode_enable(enable); }
extern "C" int bgtq_profile_decode_read(double *ms_sum, int *count)
{
    if (!ms_sum || !count) FAIL(BGTQ_EINVAL, "bgtq_profile_decode_read: null pointer");
    return profile_decode_read(ms_sum, count);
}

extern "C" int bgtq_decode_attention_layers(const bgtq_layout *lay, int layer0, int n_layers,
                                            const void *cache, const void *q, const int32_t *seq_len,
                                            int batch, int64_t max_tokens, float softmax_scale,
                                            void *out, void *workspace, size_t workspace_bytes,
                                            void *stream)
{
    if (!lay || !cache || !q || !seq_len || !out || !workspace) FAIL(BGTQ_EINVAL, "bgtq_decode_attention: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_decode_attention: layer range");
    if (batch <= 0 || max_tokens <= 0) FAIL(BGTQ_EINVAL, "bgtq_decode_attention: batch/max_tokens");
    if (!(softmax_scale > 0.0f) || std::isinf(softmax_scale)) FAIL(BGTQ_EINVAL, "bgtq_decode_attention: softmax_scale must be finite and > 0");
    if (workspace_bytes < decode_ws_any(lay, batch, n_layers)) FAIL(BGTQ_EWORKSPACE, "bgtq_decode_attention: workspace too small");
    return launch_decode_any(lay, layer0, n_layers, cache, q, seq_len, batch, max_tokens, softmax_scale,
                             out, workspace, workspace_bytes, nullptr, (cudaStream_t)stream);
}

extern "C" int bgtq_decode_attention(const bgtq_layout *lay, int layer, const void *cache, const void *q,
                                     const int32_t *seq_len, int batch, int64_t max_tokens,
                                     float softmax_scale, void *out, void *workspace,
                                     size_t workspace_bytes, void *stream)
{
    return bgtq_decode_attention_layers(lay, layer, 1, cache, q, seq_len, batch, max_tokens,
                                        softmax_scale, out, workspace, workspace_bytes, stream);
}

extern "C" int bgtq_decode_attention_protected(const bgtq_layout *lay, int layer0, int n_layers, const void *cache,
                                               const void *q, const int32_t *seq_len, int batch, int64_t max_tokens,
                                               float softmax_scale, const void *win_k, const void *win_v, int n_sink,
                                               int n_recent, void *out, void *workspace, size_t workspace_bytes,
                                               void *stream)
{
    if (!lay || !cache || !q || !seq_len || !out || !workspace || !win_k || !win_v) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_protected: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_protected: layer range");
    if (batch <= 0 || max_tokens <= 0) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_protected: batch/max_tokens");
    if (!(softmax_scale > 0.0f) || std::isinf(softmax_scale)) FAIL(BGTQ_EINVAL, "bgtq_decode_attention_protected: softmax_scale must be finite and > 0");
    if (n_sink < 0 || n_recent < 0 || n_sink >= BGTQ_TILE_TOKENS || n_sink + n_recent < 1 || n_sink + n_recent > 1024)
        FAIL(BGTQ_EINVAL, "bgtq_decode_attention_protected: need 0 <= n_sink < 128, n_recent >= 0, 1 <= n_sink + n_recent <= 1024");
    if (workspace_bytes < decode_ws_any(lay, batch, n_layers)) FAIL(BGTQ_EWORKSPACE, "bgtq_decode_attention_protected: workspace too small");
    const size_t per_layer = (size_t)batch * lay->n_kv_heads * (size_t)(n_sink + n_recent) * lay->d_h;   // fp16 elements
    const Window win = {(const uint16_t *)win_k + (size_t)layer0 * per_layer, (const uint16_t *)win_v + (size_t)layer0 * per_layer,
                        n_sink, n_recent};
    return launch_decode_any(lay, layer0, n_layers, cache, q, seq_len, batch, max_tokens, softmax_scale, out, workspace,
                             workspace_bytes, nullptr, (cudaStream_t)stream, &win);
}

extern "C" size_t bgtq_window_bytes(const bgtq_layout *lay, int batch, int n_sink, int n_recent)
{
    if (!lay || batch <= 0 || n_sink < 0 || n_recent < 0) return 0;
    return (size_t)lay->n_layers * batch * lay->n_kv_heads * (size_t)(n_sink + n_recent) * lay->d_h * 2;
}

extern "C" int bgtq_window_append(const bgtq_layout *lay, int layer0, int n_layers, const void *k_new, const void *v_new,
                                  int dt, int batch, int n_new, const int32_t *seq_len, int64_t max_tokens, void *win_k,
                                  void *win_v, int n_sink, int n_recent, void *stream)
{
    if (max_tokens <= 0) FAIL(BGTQ_EINVAL, "bgtq_window_append: max_tokens");
    if (n_sink >= BGTQ_TILE_TOKENS || n_sink + n_recent > 1024)
        FAIL(BGTQ_EINVAL, "bgtq_window_append: need 0 <= n_sink < 128, 1 <= n_sink + n_recent <= 1024");
    if (!lay || !k_new || !v_new || !seq_len || !win_k || !win_v) FAIL(BGTQ_EINVAL, "bgtq_window_append: null pointer");
    if (layer0 < 0 || n_layers <= 0 || layer0 + n_layers > lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_window_append: layer range");
    if (dt != BGTQ_F32 && dt != BGTQ_BF16) FAIL(BGTQ_EINVAL, "bgtq_window_append: dtype");
    if (batch <= 0 || n_new <= 0 || n_sink < 0 || n_recent < 0 || n_sink + n_recent < 1) FAIL(BGTQ_EINVAL, "bgtq_window_append: batch/n_new/window");
    const size_t per_layer = (size_t)batch * lay->n_kv_heads * (size_t)(n_sink + n_recent) * lay->d_h;
    return launch_window_append(k_new, v_new, dt, n_layers, batch, n_new, lay->n_kv_heads, seq_len, max_tokens,
                                (uint16_t *)win_k + (size_t)layer0 * per_layer, (uint16_t *)win_v + (size_t)layer0 * per_layer,
                                n_sink, n_recent, (cudaStream_t)stream);
}

extern "C" size_t bgtq_prefill_workspace_bytes(const bgtq_layout *lay, int batch, int n_q)
{
    if (!lay || batch <= 0 || n_q <= 0) return 0;
    return prefill_ws_bytes(lay, batch, n_q);
}

extern "C" int bgtq_prefill_attention(const bgtq_layout *lay, int layer, const void *cache, const void *q,
                                      const int32_t *seq_len, int batch, int n_q, int64_t max_tokens,
                                      float softmax_scale, void *out, void *workspace, size_t workspace_bytes,
                                      void *stream)
{
    if (!lay || !cache || !q || !seq_len || !out || !workspace) FAIL(BGTQ_EINVAL, "bgtq_prefill_attention: null pointer");
    if (layer < 0 || layer >= lay->n_layers) FAIL(BGTQ_EINVAL, "bgtq_prefill_attention: layer out of range");
    if (lay->format != BGTQ_FORMAT_V1 || lay->cb_exact || lay->v_grouped) FAIL(BGTQ_EINVAL, "bgtq_prefill_attention: built for BGTQ_FORMAT_V1 layouts with the shared codebooks and one V group per head only");
    if (batch <= 0 || n_q <= 0 || max_tokens <= 0 || n_q > max_tokens) FAIL(BGTQ_EINVAL, "bgtq_prefill_attention: batch/n_q/max_tokens");
    if (!(softmax_scale > 0.0f) || std::isinf(softmax_scale)) FAIL(BGTQ_EINVAL, "bgtq_prefill_attention: softmax_scale");
    return launch_prefill(lay, layer, cache, q, seq_len, batch, n_q, max_tokens, softmax_scale, out, workspace,
                          workspace_bytes, (cudaStream_t)stream);
}

extern "C" size_t bgtq_fp16_workspace_bytes(int batch, int n_layers, int n_kv_heads)
{
    if (batch <= 0 || n_layers <= 0 || n_kv_heads <= 0) return 0;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms = 256;
    return fp16_ws_bytes(sms, batch, n_layers, n_kv_heads);
}

extern "C" int bgtq_fp16_decode_attention(int n_layers, int batch, int n_q_heads, int n_kv_heads, int d_h,
                                          const void *k_cache, const void *v_cache, const void *q,
                                          const int32_t *seq_len, int64_t max_tokens, float softmax_scale,
                                          void *out, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!k_cache || !v_cache || !q || !seq_len || !out || !workspace) FAIL(BGTQ_EINVAL, "bgtq_fp16_decode_attention: null pointer");
    if (d_h != kDh) FAIL(BGTQ_EINVAL, "bgtq_fp16_decode_attention: d_h must be 128");
    if (n_layers <= 0 || batch <= 0 || n_kv_heads <= 0 || n_q_heads % n_kv_heads || n_q_heads / n_kv_heads > 8 || n_q_heads <= 0)
        FAIL(BGTQ_EINVAL, "bgtq_fp16_decode_attention: bad shape (GQA group <= 8)");
    if (max_tokens <= 0 || max_tokens % BGTQ_TILE_TOKENS) FAIL(BGTQ_EINVAL, "bgtq_fp16_decode_attention: max_tokens must be a positive multiple of 128");
    if (!(softmax_scale > 0.0f)) FAIL(BGTQ_EINVAL, "bgtq_fp16_decode_attention: softmax_scale");
    return launch_fp16_decode(n_layers, batch, n_q_heads, n_kv_heads, k_cache, v_cache, q, seq_len, max_tokens,
                              softmax_scale, out, workspace, workspace_bytes, (cudaStream_t)stream);
}

extern "C" int bgtq_debug_decode_unit(int b, const uint32_t *words, float *values)
{
    if (b < 1 || b > BGTQ_MAX_WIDTH || !words || !values) FAIL(BGTQ_EINVAL, "bgtq_debug_decode_unit: bad argument");
    return debug_decode_unit(b, words, values);
}
