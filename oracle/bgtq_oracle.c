/*
 * bgtq_oracle.c -- plain, slow, fp64 CPU oracle for the Block-GTQ hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or generator with the CUDA path under paper_2606_24033_b200/.
 *
 * Every function follows a passage of /root/reference/PAPER.md (cited as PAPER.md:<line>)
 * or, where the paper is silent, a numbered reading "Qn" listed in DESIGN.md.
 * Parity pins: tests/test_oracle_*.py (-m "not gpu").  Status per function:
 *   orc_rope               pinned (block-sum identity PAPER.md:43, Eq. 2)
 *   orc_block_energy       pinned (closed form 2*var, AM-GM PAPER.md:63, Jensen PAPER.md:614)
 *   orc_allocate_*         pinned (brute force = Thm. 1; heap == linear)
 *   orc_quantize_group /
 *   orc_dequantize_group   pinned to the rate law PAPER.md:49 and to brute-force nearest
 *                          centroid; "parity unpinned" against the AUTHORS' codebook /
 *                          rotation / layout (the paper prints none) -- see DESIGN.md.
 *   orc_put_field / get    pinned (round trip, byte accounting PAPER.md:837, hand-worked tests/golden/layout_*.txt)
 *   orc_*_v2 (BGTQ-v2)     pinned (hand-worked tests/golden/layout_fields_v2.txt, layout_region_v2.txt; bijection; round trip)
 *   orc_f64_to_f16_bits /
 *   orc_f16_bits_to_f64    pinned to IEEE binary16 via numpy.float16 (every value, every midpoint, saturation)
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
 * -ffp-contract=off matters: every rounding below is the one written.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ fp16 <-> fp64 */

/* IEEE binary16 round-to-nearest-even of a finite double, saturating to 65504
 * (Q10: fp16 norm, RNE, saturate).  Done on the bits, no _Float16. */
uint16_t orc_f64_to_f16_bits(double x)
{
    uint16_t sign = 0;
    if (signbit(x)) { sign = 0x8000u; x = -x; }
    if (x != x) return (uint16_t)(sign | 0x7E00u);
    if (x >= 65520.0) return (uint16_t)(sign | 0x7BFFu);          /* saturate (65520 rounds up) */
    if (x < ldexp(1.0, -25)) return sign;                          /* < half of smallest subnormal */
    int e;
    double f = frexp(x, &e);          /* x = f * 2^e, f in [0.5,1) */
    int E = e - 1;                    /* x = (2f) * 2^E, 2f in [1,2) */
    double scaled;
    int biased;
    if (E < -14) {                    /* subnormal: units of 2^-24 */
        scaled = ldexp(x, 24);
        biased = 0;
    } else {
        scaled = ldexp(2.0 * f, 10);  /* in [1024, 2048) */
        biased = E + 15;
    }
    double fl = floor(scaled);
    double rem = scaled - fl;
    uint32_t q = (uint32_t)fl;
    if (rem > 0.5 || (rem == 0.5 && (q & 1u))) q += 1u;
    uint32_t bits;
    if (biased == 0) bits = q;                       /* may carry into exponent 1: correct */
    else bits = ((uint32_t)biased << 10) + (q - 1024u);  /* carry of q==2048 bumps exponent */
    if (bits >= 0x7C00u) bits = 0x7BFFu;
    return (uint16_t)(sign | bits);
}

double orc_f16_bits_to_f64(uint16_t h)
{
    int s = (h >> 15) & 1, e = (h >> 10) & 31, m = h & 1023;
    double v;
    if (e == 0) v = ldexp((double)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexp(1.0 + (double)m / 1024.0, e - 15);
    return s ? -v : v;
}

/* ------------------------------------------------------------------ RoPE (harness side) */

/* Block i of a head = coordinates (a(i), b(i)).  pairing 0: (i, i+d/2); 1: (2i, 2i+1)
 * (Q1).  theta_i = base^(-2i/d_h), R(phi) = [[cos,-sin],[sin,cos]] (Q2);
 * x^R_t = R_t x with R_t = diag(R(t*theta_i)).                       */
static void pair_index(int d_h, int pairing, int i, int *a, int *b)
{
    if (pairing == 0) { *a = i; *b = i + d_h / 2; }
    else { *a = 2 * i; *b = 2 * i + 1; }
}

void orc_rope(const double *x, long n, int n_heads, int d_h, const double *pos, double base,
              int pairing, double *out)
{
    int L = d_h / 2;
    for (long t = 0; t < n; ++t)
        for (int h = 0; h < n_heads; ++h) {
            const double *xi = x + ((size_t)t * n_heads + h) * d_h;
            double *o = out + ((size_t)t * n_heads + h) * d_h;
            for (int i = 0; i < L; ++i) {
                int a, b;
                pair_index(d_h, pairing, i, &a, &b);
                double theta = pow(base, -2.0 * (double)i / (double)d_h);
                double phi = pos[t] * theta;
                double c = cos(phi), s = sin(phi);
                o[a] = c * xi[a] - s * xi[b];
                o[b] = s * xi[a] + c * xi[b];
            }
        }
}

/* ------------------------------------------------------------------ block energy */

/* Eq. 4, Alg. 2 lines 6-7: two plain means.
 *   Eq[h][i] = 1/(N_q*G) sum_t sum_{g in G(h)} ||q_{g,t}^(i)||^2    (square THEN average,
 *   Ek[h][i] = 1/N_k     sum_t ||k_{h,t}^(i)||^2                     PAPER.md:614)
 * G(h) = {h*G .. h*G+G-1}; N_q and N_k independent (Q15).  Sequential fp64 sums. */
void orc_block_energy(const double *q, long n_q, int n_q_heads, const double *k, long n_k,
                      int n_kv_heads, int d_h, int pairing, double *Eq, double *Ek)
{
    int L = d_h / 2, G = n_q_heads / n_kv_heads;
    for (int h = 0; h < n_kv_heads; ++h)
        for (int i = 0; i < L; ++i) {
            int a, b;
            pair_index(d_h, pairing, i, &a, &b);
            double sq = 0.0;
            for (long t = 0; t < n_q; ++t)
                for (int g = h * G; g < h * G + G; ++g) {
                    const double *v = q + ((size_t)t * n_q_heads + g) * d_h;
                    sq += v[a] * v[a] + v[b] * v[b];
                }
            double sk = 0.0;
            for (long t = 0; t < n_k; ++t) {
                const double *v = k + ((size_t)t * n_kv_heads + h) * d_h;
                sk += v[a] * v[a] + v[b] * v[b];
            }
            Eq[h * L + i] = n_q > 0 ? sq / ((double)n_q * (double)G) : 0.0;
            Ek[h * L + i] = n_k > 0 ? sk / (double)n_k : 0.0;
        }
}

/* Score kinds.  0 qk_avg (Eq. 1/4), 1 qk_max, 2 qk_product, 3 k_only, 4 q_only */
double orc_score(double eq, double ek, int kind)
{
    switch (kind) {
    case 0: return 0.5 * (eq + ek);
    case 1: return eq > ek ? eq : ek;
    case 2: return sqrt(eq * ek);
    case 3: return ek;
    default: return eq;
    }
}

/* ------------------------------------------------------------------ Algorithm 1 */

/* key of block i at width b: Delta_i = 3/4 * s_i * 4^-b.  ldexp is exact. */
static double gain_key(double s, int b) { return 0.75 * ldexp(s, -2 * b); }

/* Alg. 1 with a linear arg-max; ties -> smallest i (Q4); zero scores get key 0 and
 * so receive bits only after positive-gain blocks saturate, in index order (Q5).
 * gains (optional) records the popped Delta sequence.  Returns 0, or -1 if B infeasible. */
int orc_allocate_linear(const double *s, int L, int b_min, int b_max, int B, uint8_t *bits,
                        double *gains)
{
    if (B < L * b_min || B > L * b_max) return -1;
    for (int i = 0; i < L; ++i) bits[i] = (uint8_t)b_min;                 /* line 1 */
    int extra = B - L * b_min;                                            /* line 2 */
    for (int step = 0; step < extra; ++step) {                            /* line 4 */
        int best = -1;
        double bestkey = -1.0;
        for (int i = 0; i < L; ++i) {
            if (bits[i] >= b_max) continue;                               /* line 3 / 7 */
            double key = gain_key(s[i], bits[i]);
            if (key > bestkey) { bestkey = key; best = i; }               /* strict: smallest i */
        }
        if (best < 0) break;
        if (gains) gains[step] = bestkey;
        bits[best] += 1;                                                  /* line 6 */
    }
    return 0;
}

/* Alg. 1 verbatim with a binary max-heap.  Order: larger key first,
 * equal keys -> smaller index first.  Must equal orc_allocate_linear (tested). */
typedef struct { double key; int idx; } heap_item;
static int heap_before(heap_item a, heap_item b)
{
    return a.key > b.key || (a.key == b.key && a.idx < b.idx);
}
static void heap_push(heap_item *h, int *n, heap_item it)
{
    int i = (*n)++;
    h[i] = it;
    while (i > 0) {
        int p = (i - 1) / 2;
        if (!heap_before(h[i], h[p])) break;
        heap_item t = h[i]; h[i] = h[p]; h[p] = t;
        i = p;
    }
}
static heap_item heap_pop(heap_item *h, int *n)
{
    heap_item top = h[0];
    h[0] = h[--(*n)];
    int i = 0;
    for (;;) {
        int l = 2 * i + 1, r = l + 1, m = i;
        if (l < *n && heap_before(h[l], h[m])) m = l;
        if (r < *n && heap_before(h[r], h[m])) m = r;
        if (m == i) break;
        heap_item t = h[i]; h[i] = h[m]; h[m] = t;
        i = m;
    }
    return top;
}
int orc_allocate_heap(const double *s, int L, int b_min, int b_max, int B, uint8_t *bits)
{
    if (B < L * b_min || B > L * b_max) return -1;
    heap_item *heap = (heap_item *)malloc(sizeof(heap_item) * (size_t)(L > 0 ? L : 1));
    int n = 0;
    for (int i = 0; i < L; ++i) bits[i] = (uint8_t)b_min;
    int extra = B - L * b_min;
    if (b_min < b_max)
        for (int i = 0; i < L; ++i) {
            heap_item it = { gain_key(s[i], b_min), i };
            heap_push(heap, &n, it);
        }
    while (extra > 0 && n > 0) {
        heap_item top = heap_pop(heap, &n);
        bits[top.idx] += 1;
        extra -= 1;
        if (bits[top.idx] < b_max) {
            heap_item it = { gain_key(s[top.idx], bits[top.idx]), top.idx };
            heap_push(heap, &n, it);
        }
    }
    free(heap);
    return 0;
}

/* J(b) = sum_i s_i 4^-b_i */
double orc_objective(const double *s, const uint8_t *bits, int L)
{
    double J = 0.0;
    for (int i = 0; i < L; ++i) J += ldexp(s[i], -2 * (int)bits[i]);
    return J;
}

/* ------------------------------------------------------------------ TQ-MSE (BGTQ-v1) */

/* Quantise one same-width group (PAPER.md:49 normalise -> rotate -> scalar-quantise -> keep
 * radius; PAPER.md:108 one encoder per group).  DESIGN.md "Oracle step 5", verbatim:
 *   ss = fma chain over j;  r = sqrt(ss);  sigma = r / sqrt((double)m);
 *   z_j = fma chain over k of Pi[j][k] * x_k;
 *   idx_j = #{ k : z_j > tau_k * sigma },  tau_k = (C[k] + C[k+1]) / 2   (strict >: Q11)
 *   h = fp16_rne(r), saturating.
 * x: m doubles (exact up-conversions of the fp32/bf16 inputs); Pi: m*m fp32 row-major;
 * C: 2^b ascending levels (fp16-representable doubles).  b >= 1.                           */
void orc_quantize_group(const double *x, int m, const float *Pi, const double *C, int b,
                        uint8_t *idx, uint16_t *h_bits, double *r_out)
{
    double ss = 0.0;
    for (int j = 0; j < m; ++j) ss = fma(x[j], x[j], ss);
    double r = sqrt(ss);
    double sigma = r / sqrt((double)m);
    int nlev = 1 << b;
    for (int j = 0; j < m; ++j) {
        double z = 0.0;
        for (int k = 0; k < m; ++k) z = fma((double)Pi[(size_t)j * m + k], x[k], z);
        int count = 0;
        for (int k = 0; k + 1 < nlev; ++k) {
            double tau = (C[k] + C[k + 1]) / 2.0;
            double thr = tau * sigma;
            if (z > thr) count += 1;
        }
        idx[j] = (uint8_t)count;
    }
    *h_bits = orc_f64_to_f16_bits(r);
    if (r_out) *r_out = r;
}

/* Dequantise:  xhat_k = (h / sqrt(m)) * sum_j Pi[j][k] * C[idx_j]. */
void orc_dequantize_group(const uint8_t *idx, int m, uint16_t h_bits, const float *Pi,
                          const double *C, double *xhat)
{
    double h = orc_f16_bits_to_f64(h_bits);
    double scale = h / sqrt((double)m);
    for (int k = 0; k < m; ++k) {
        double acc = 0.0;
        for (int j = 0; j < m; ++j) acc += (double)Pi[(size_t)j * m + k] * C[idx[j]];
        xhat[k] = scale * acc;
    }
}

/* ------------------------------------------------------------------ physical layout BGTQ-v1
 * DESIGN.md section "Packed cache layout" is the specification; this is its independent
 * restatement.  A "unit" is b 32-bit words W[0..b-1] holding 32 b-bit fields ("slots").      */

/* width-4 fields are stored sign-magnitude: idx>=8 -> (s=0, mag=idx-8); idx<8 -> (s=1, mag=7-idx) */
static unsigned recode4(unsigned idx) { return idx >= 8 ? (idx - 8) : (8u | (7u - idx)); }
static unsigned decode4(unsigned f) { return (f & 8u) ? (7u - (f & 7u)) : ((f & 7u) + 8u); }

static void setbit(uint32_t *W, int word, int bit, unsigned v)
{
    W[word] = (W[word] & ~(1u << bit)) | ((v & 1u) << bit);
}
static unsigned getbit(const uint32_t *W, int word, int bit) { return (W[word] >> bit) & 1u; }

/* position of bit `bit` of the mag3 field of slot k in the 3-word "nibble + spare" scheme */
static void mag3_pos(int k, int bit, int *word, int *pos)
{
    if (k < 24) { *word = k >> 3; *pos = 4 * (k & 7) + bit; }
    else { *word = bit; *pos = 4 * (k - 24) + 3; }
}

void orc_put_field(uint32_t *W, int b, int k, unsigned idx)
{
    int word, pos;
    switch (b) {
    case 1:   /* slot 2j+e at bit (15-j)+16e */
        setbit(W, 0, (15 - (k >> 1)) + 16 * (k & 1), idx);
        break;
    case 2: { /* word k>>4; kk=k&15, Q=kk>>2, e=kk&3: field at 4*((Q&1)*4+e) + 2*(Q>>1) */
        int kk = k & 15, Q = kk >> 2, e = kk & 3;
        int p = 4 * ((Q & 1) * 4 + e) + 2 * (Q >> 1);
        setbit(W, k >> 4, p, idx);
        setbit(W, k >> 4, p + 1, idx >> 1);
        break;
    }
    case 3:
        for (int bit = 0; bit < 3; ++bit) { mag3_pos(k, bit, &word, &pos); setbit(W, word, pos, idx >> bit); }
        break;
    case 4: {
        unsigned f = recode4(idx);
        for (int bit = 0; bit < 3; ++bit) { mag3_pos(k, bit, &word, &pos); setbit(W, word, pos, f >> bit); }
        setbit(W, 3, 8 * (k & 3) + 7 - (k >> 2), f >> 3);   /* slot 4Q+e: bit 8e+7-Q */
        break;
    }
    default:  /* b = 5..8: field occupies bits [b*k, b*k+b) of the little-endian stream */
        for (int bit = 0; bit < b; ++bit) {
            int s = b * k + bit;
            setbit(W, s >> 5, s & 31, idx >> bit);
        }
    }
}

unsigned orc_get_field(const uint32_t *W, int b, int k)
{
    int word, pos;
    unsigned f = 0;
    switch (b) {
    case 1:
        return getbit(W, 0, (15 - (k >> 1)) + 16 * (k & 1));
    case 2: {
        int kk = k & 15, Q = kk >> 2, e = kk & 3;
        int p = 4 * ((Q & 1) * 4 + e) + 2 * (Q >> 1);
        return getbit(W, k >> 4, p) | (getbit(W, k >> 4, p + 1) << 1);
    }
    case 3:
        for (int bit = 0; bit < 3; ++bit) { mag3_pos(k, bit, &word, &pos); f |= getbit(W, word, pos) << bit; }
        return f;
    case 4:
        for (int bit = 0; bit < 3; ++bit) { mag3_pos(k, bit, &word, &pos); f |= getbit(W, word, pos) << bit; }
        f |= getbit(W, 3, 8 * (k & 3) + 7 - (k >> 2)) << 3;
        return decode4(f);
    default:
        for (int bit = 0; bit < b; ++bit) {
            int s = b * k + bit;
            f |= getbit(W, s >> 5, s & 31) << bit;
        }
        return f;
    }
}

/* norm slot of token tau (0..127) inside a 128-entry fp16 norm row: g*16 + i*2 + p,
 * with i = tau>>4, g = tau&7, p = (tau>>3)&1.                                              */
static int norm_slot(int tau) { return (tau & 7) * 16 + (tau >> 4) * 2 + ((tau >> 3) & 1); }

/* Pack (or with unpack!=0: unpack) tokens [t0, t1) of ONE (sequence, layer, KV head) region.
 *   region   : n_tiles * tile_stride bytes, tile = [K codes | K norms | V norms | V codes]
 *   n_groups, gb[g] (width, ascending, >=1), gm[g] (coords in group, even)
 *   kidx     : [T][kdim] K codes, grouped coordinate order (groups concatenated), kdim = sum gm
 *   knorm    : [T][n_groups] fp16 bits;  vidx: [T][d_h];  vnorm: [T]
 * Only the fields of tokens in [t0,t1) are touched; everything else is preserved.           */
void orc_pack_region_kv(uint8_t *region, long tile_stride, int n_groups, const int *gb, const int *gm,
                        int d_h, int n_vgroups, const int *vgb, const int *vgm, long t0, long t1,
                        uint8_t *kidx, uint16_t *knorm, uint8_t *vidx, uint16_t *vnorm, int unpack);

void orc_pack_region(uint8_t *region, long tile_stride, int n_groups, const int *gb, const int *gm,
                     int d_h, int b_v, long t0, long t1, uint8_t *kidx, uint16_t *knorm,
                     uint8_t *vidx, uint16_t *vnorm, int unpack)
{
    /* V: one group of all d_h coordinates at width b_v */
    orc_pack_region_kv(region, tile_stride, n_groups, gb, gm, d_h, 1, &b_v, &d_h, t0, t1, kidx, knorm, vidx, vnorm, unpack);
}

/* The general form (V-side groups, reading Q19): V group gv has width vgb[gv] (ascending) and vgm[gv]
 * coordinates (a multiple of 16: whole V blocks); tile = [K codes | K norms | V norms (n_vgroups rows) | V codes
 * (groups in order, 16 * vgm * vgb bytes each)].
 *   vidx  : [T][d_h] V codes in grouped V order (groups concatenated);  vnorm: [T][n_vgroups]                     */
void orc_pack_region_kv(uint8_t *region, long tile_stride, int n_groups, const int *gb, const int *gm,
                        int d_h, int n_vgroups, const int *vgb, const int *vgm, long t0, long t1,
                        uint8_t *kidx, uint16_t *knorm, uint8_t *vidx, uint16_t *vnorm, int unpack)
{
    int kdim = 0;
    long kcode_bytes = 0;
    for (int g = 0; g < n_groups; ++g) { kdim += gm[g]; kcode_bytes += 16L * gm[g] * gb[g]; }
    long knorm_off = kcode_bytes;
    long vnorm_off = knorm_off + 256L * n_groups;
    long vcode_off = vnorm_off + 256L * n_vgroups;
    for (long t = t0; t < t1; ++t) {
        uint8_t *tile = region + (t >> 7) * tile_stride;
        int tau = (int)(t & 127);
        int i = tau >> 4, g8 = tau & 7, p = (tau >> 3) & 1;
        /* ---- K codes: group -> half-step j (8 coords) -> lane (g8, c) -> slot i*4+p*2+q */
        long goff = 0;
        int ubase = 0;
        for (int g = 0; g < n_groups; ++g) {
            int b = gb[g], m = gm[g];
            for (int u = 0; u < m; ++u) {
                int j = u >> 3, v = u & 7, c = v >> 1, q = v & 1;
                int real = m - 8 * j >= 8 ? 8 : m - 8 * j;      /* coords in this half-step */
                int nc = real / 2;                               /* lanes per g8 row */
                int lanes = 8 * nc;
                long unit = goff + (long)j * b * 128;           /* earlier half-steps are full */
                int lane = g8 * nc + c;
                int slot = i * 4 + p * 2 + q;
                uint32_t W[8];
                for (int w = 0; w < b; ++w)
                    memcpy(&W[w], tile + unit + 4L * ((long)w * lanes + lane), 4);
                if (unpack) kidx[(size_t)t * kdim + ubase + u] = (uint8_t)orc_get_field(W, b, slot);
                else {
                    orc_put_field(W, b, slot, kidx[(size_t)t * kdim + ubase + u]);
                    for (int w = 0; w < b; ++w)
                        memcpy(tile + unit + 4L * ((long)w * lanes + lane), &W[w], 4);
                }
            }
            /* ---- K norm of this group */
            uint8_t *np_ = tile + knorm_off + 256L * g + 2L * norm_slot(tau);
            if (unpack) memcpy(&knorm[(size_t)t * n_groups + g], np_, 2);
            else memcpy(np_, &knorm[(size_t)t * n_groups + g], 2);
            goff += 16L * m * b;
            ubase += m;
        }
        /* ---- V: per group its norm, then its codes.  Inside a group, grouped coordinate u -> J=u>>4, g=u&7,
         *      rho=(u>>3)&1; token -> kappa=tau>>4, c=(tau&7)>>1, e=tau&1, o=(tau>>3)&1; unit J*2+rho of the group,
         *      lane g*4+c, slot kappa*4+o*2+e */
        long vgoff = 0;
        int vbase = 0;
        for (int gv = 0; gv < n_vgroups; ++gv) {
            int b_v = vgb[gv], mv = vgm[gv];
            uint8_t *np_ = tile + vnorm_off + 256L * gv + 2L * norm_slot(tau);
            if (unpack) memcpy(&vnorm[(size_t)t * n_vgroups + gv], np_, 2);
            else memcpy(np_, &vnorm[(size_t)t * n_vgroups + gv], 2);
            for (int u = 0; u < mv; ++u) {
                int J = u >> 4, g = u & 7, rho = (u >> 3) & 1;
                int kappa = tau >> 4, c = (tau & 7) >> 1, e = tau & 1, o = (tau >> 3) & 1;
                long unit = vcode_off + vgoff + (long)(J * 2 + rho) * b_v * 128;
                int lane = g * 4 + c, slot = kappa * 4 + o * 2 + e;
                uint32_t W[8];
                for (int w = 0; w < b_v; ++w) memcpy(&W[w], tile + unit + 4L * (w * 32 + lane), 4);
                if (unpack) vidx[(size_t)t * d_h + vbase + u] = (uint8_t)orc_get_field(W, b_v, slot);
                else {
                    orc_put_field(W, b_v, slot, vidx[(size_t)t * d_h + vbase + u]);
                    for (int w = 0; w < b_v; ++w) memcpy(tile + unit + 4L * (w * 32 + lane), &W[w], 4);
                }
            }
            vgoff += 16L * mv * b_v;
            vbase += mv;
        }
    }
}

/* ------------------------------------------------------------------ physical layout BGTQ-v2 ("row order")
 * DESIGN.md section 4b is the specification; this is its independent restatement.
 * A tile is still 128 tokens, [K codes | K norms | V norms | V codes], but a code word now belongs to ONE row of the
 * tensor-core operand: token tau = 32*w + l (quadrant w, lane l) owns its K codes, dimension d = 32*w + l owns its V
 * codes.  A "chunk" is up to 32 slots of one row: K chunk u of group g = grouped coordinates 32u .. 32u+r-1 of the
 * group (r = min(32, m - 32u)); V chunk c of dimension d = tokens 32c .. 32c+31.  A chunk stores nw(b, r) 32-bit
 * words per lane, plane-major (word j of lane l at byte 4*(j*32 + l)).
 *   slot -> bits: b = 1: slot 4Q+e at word 0 bit 8e+7-Q;  b = 2, 3, >= 5: as BGTQ-v1 (orc_put_field);
 *                 b = 4: magnitudes as b = 3 in words 0 .. nwm-1, sign of slot 4Q+e at word nwm, bit 8e+7-Q
 *   nw(b, r):     b = 1: 1;  b = 2: ceil(r/16);  b = 3: nwm = min(3, ceil(r/8));  b = 4: nwm + 1;  b >= 5: ceil(r*b/32)
 * Norm rows are in natural token order (token tau at entry tau).                                                     */
int orc_chunk_words_v2(int b, int r)
{
    int nwm = r > 24 ? 3 : (r + 7) / 8;
    switch (b) {
    case 1: return 1;
    case 2: return (r + 15) / 16;
    case 3: return nwm;
    case 4: return nwm + 1;
    default: return (r * b + 31) / 32;
    }
}

void orc_put_field_v2(uint32_t *W, int b, int r, int k, unsigned idx)
{
    int word, pos;
    if (b == 1) setbit(W, 0, 8 * (k & 3) + 7 - (k >> 2), idx);
    else if (b == 4) {
        unsigned f = recode4(idx);
        int nwm = r > 24 ? 3 : (r + 7) / 8;
        for (int bit = 0; bit < 3; ++bit) { mag3_pos(k, bit, &word, &pos); setbit(W, word, pos, f >> bit); }
        setbit(W, nwm, 8 * (k & 3) + 7 - (k >> 2), f >> 3);
    } else orc_put_field(W, b, k, idx);
}

unsigned orc_get_field_v2(const uint32_t *W, int b, int r, int k)
{
    int word, pos;
    unsigned f = 0;
    if (b == 1) return getbit(W, 0, 8 * (k & 3) + 7 - (k >> 2));
    if (b == 4) {
        int nwm = r > 24 ? 3 : (r + 7) / 8;
        for (int bit = 0; bit < 3; ++bit) { mag3_pos(k, bit, &word, &pos); f |= getbit(W, word, pos) << bit; }
        f |= getbit(W, nwm, 8 * (k & 3) + 7 - (k >> 2)) << 3;
        return decode4(f);
    }
    return orc_get_field(W, b, k);
}

/* bytes of the K codes of ONE quadrant (32 tokens) of a tile */
long orc_kquad_bytes_v2(int n_groups, const int *gb, const int *gm)
{
    long words = 0;
    for (int g = 0; g < n_groups; ++g)
        for (int u = 0; 32 * u < gm[g]; ++u) {
            int r = gm[g] - 32 * u >= 32 ? 32 : gm[g] - 32 * u;
            words += orc_chunk_words_v2(gb[g], r);
        }
    return 128L * words;
}

/* Same contract as orc_pack_region, BGTQ-v2 layout. */
void orc_pack_region_v2(uint8_t *region, long tile_stride, int n_groups, const int *gb, const int *gm,
                        int d_h, int b_v, long t0, long t1, uint8_t *kidx, uint16_t *knorm,
                        uint8_t *vidx, uint16_t *vnorm, int unpack)
{
    int kdim = 0;
    for (int g = 0; g < n_groups; ++g) kdim += gm[g];
    long kq = orc_kquad_bytes_v2(n_groups, gb, gm);
    long knorm_off = 4 * kq;
    long vnorm_off = knorm_off + 256L * n_groups;
    long vcode_off = vnorm_off + 256L;
    for (long t = t0; t < t1; ++t) {
        uint8_t *tile = region + (t >> 7) * tile_stride;
        int tau = (int)(t & 127), w = tau >> 5, l = tau & 31;
        /* ---- K codes: quadrant w -> group -> chunk u -> word planes; lane l = token, slot = coordinate */
        long coff = (long)w * kq;
        int ubase = 0;
        for (int g = 0; g < n_groups; ++g) {
            int b = gb[g], m = gm[g];
            for (int u = 0; 32 * u < m; ++u) {
                int r = m - 32 * u >= 32 ? 32 : m - 32 * u;
                int nw = orc_chunk_words_v2(b, r);
                uint32_t W[8];
                for (int j = 0; j < nw; ++j) memcpy(&W[j], tile + coff + 4L * (j * 32 + l), 4);
                for (int s = 0; s < r; ++s) {
                    size_t src = (size_t)t * kdim + ubase + 32 * u + s;
                    if (unpack) kidx[src] = (uint8_t)orc_get_field_v2(W, b, r, s);
                    else orc_put_field_v2(W, b, r, s, kidx[src]);
                }
                if (!unpack)
                    for (int j = 0; j < nw; ++j) memcpy(tile + coff + 4L * (j * 32 + l), &W[j], 4);
                coff += 128L * nw;
            }
            uint8_t *np_ = tile + knorm_off + 256L * g + 2L * tau;
            if (unpack) memcpy(&knorm[(size_t)t * n_groups + g], np_, 2);
            else memcpy(np_, &knorm[(size_t)t * n_groups + g], 2);
            ubase += m;
        }
        /* ---- V norm */
        {
            uint8_t *np_ = tile + vnorm_off + 2L * tau;
            if (unpack) memcpy(&vnorm[t], np_, 2);
            else memcpy(np_, &vnorm[t], 2);
        }
        /* ---- V codes: dimension d = 32*wq + lane; chunk c = tau>>5; slot = tau&31 */
        for (int d = 0; d < d_h; ++d) {
            int wq = d >> 5, lane = d & 31;
            long unit = vcode_off + (long)((wq * 4 + w) * b_v) * 128;
            uint32_t W[8];
            for (int j = 0; j < b_v; ++j) memcpy(&W[j], tile + unit + 4L * (j * 32 + lane), 4);
            if (unpack) vidx[(size_t)t * d_h + d] = (uint8_t)orc_get_field_v2(W, b_v, 32, l);
            else {
                orc_put_field_v2(W, b_v, 32, l, vidx[(size_t)t * d_h + d]);
                for (int j = 0; j < b_v; ++j) memcpy(tile + unit + 4L * (j * 32 + lane), &W[j], 4);
            }
        }
    }
}
