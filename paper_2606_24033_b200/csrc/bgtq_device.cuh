// bgtq_device.cuh -- device-side helpers shared by the decode kernels (bgtq_decode.cu: BGTQ-v1 mma.sync path, prefill,
// combine; bgtq_decode2.cu: BGTQ-v2 tcgen05 path).  Inline PTX wrappers, the programmatic-dependent-launch pair and the
// split-KV work partition.  Not installed.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "bgtq_internal.h"

namespace bgtq {

constexpr int kMaxWarpsPerSM = 16;
constexpr int kMaxBatch = 256;
constexpr int kPartialFloats = 8 * 130;             // (m, l, acc[128]) for 8 head slots

// ---------------------------------------------------------------- small PTX wrappers
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t s)
{
    uint32_t r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(s));
    return r;
}
__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                         uint32_t a3, uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// same with C = 0 (the zero register): starts an accumulator without a separate zero-fill
__device__ __forceinline__ void mma16816_z(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                           uint32_t a3, uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
        : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(0.f));
}
// m16n8k8 (one 8-coordinate unit): a0 = (row g8, k 2c, 2c+1), a1 = (row g8+8, ...), b0 = (k 2c, 2c+1; n g8)
__device__ __forceinline__ void mma1688(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t b0)
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(b0));
}
__device__ __forceinline__ void mma1688_z(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0)
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%7,%7,%7,%7};"
        : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3]) : "r"(a0), "r"(a1), "r"(b0), "f"(0.f));
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t x)
{
    uint32_t r;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}
__device__ __forceinline__ float fast_exp2(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi)
{
    uint32_t r;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        // (with a suspend-time hint the waiting thread is parked by the hardware until the phase completes -- or the hint,
        //  in nanoseconds, expires -- instead of re-issuing the test every few dozen clocks and stealing issue slots)
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
    } while (!done);
}
// one non-blocking test of a phase (for a thread that watches several barriers)
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    return done != 0;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}

// ---------------------------------------------------------------- programmatic dependent launch
// qfold -> decode -> combine are launched back to back on one stream.  decode and combine are launched with the
// programmatic-stream-serialization attribute: their CTAs may start while the previous kernel is still running
// (pdl_trigger in that kernel), run their prologue (LUTs, prefix sums, slot lists), and block in pdl_wait until the
// previous kernel has completed and its writes are visible.  Nothing written by a predecessor is read before pdl_wait.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---------------------------------------------------------------- work partition
// Global tile list [layer][sequence][kv head][tile]; pre[] = prefix sums of tiles per sequence.
struct Sched {
    int n_layers, batch, Hkv;
    int tiles_sum;          // sum over sequences of ceil(seq_len/128)
    int total;              // n_layers * Hkv * tiles_sum
    int n_ctas, W;          // balanced two-level split: CTA c owns [cta_lo(c), cta_lo(c+1)), its W warps split that evenly
};
__device__ __forceinline__ int cta_lo(const Sched &s, int c) { return (int)(((int64_t)c * s.total) / s.n_ctas); }
__device__ __forceinline__ int warp_lo(const Sched &s, int c, int w)
{
    const int lo = cta_lo(s, c), len = cta_lo(s, c + 1) - lo;
    return lo + (int)(((int64_t)w * len) / s.W);
}

// Protected regime: of the T cached tokens of a sequence the packed cache serves
// [n_sink, T - n_recent) only -- the first n_sink and the last n_recent tokens are attended from fp16 windows by
// window_kernel.  Number of packed tokens to scan (tokens below n_sink are masked inside tile 0); 0 when the range is empty.
__device__ __forceinline__ int64_t packed_len(int64_t T, int n_sink, int n_recent)
{
    const int64_t hi = T - n_recent;
    return hi > n_sink ? hi : 0;
}
__device__ __forceinline__ void build_prefix(const int32_t *seq_len, int batch, int64_t cap_tokens, int *pre,
                                             int n_sink = 0, int n_recent = 0)
{
    // called by one thread; batch <= kMaxBatch
    int acc = 0;
    pre[0] = 0;
    for (int b = 0; b < batch; ++b) {
        int64_t n = seq_len[b];
        n = n < 0 ? 0 : (n > cap_tokens ? cap_tokens : n);
        n = packed_len(n, n_sink, n_recent);
        acc += (int)((n + kTile - 1) / kTile);
        pre[b + 1] = acc;
    }
}

__device__ __forceinline__ Sched make_sched(int n_layers, int batch, int Hkv, const int *pre, int n_ctas, int W)
{
    Sched s;
    s.n_layers = n_layers; s.batch = batch; s.Hkv = Hkv;
    s.tiles_sum = pre[batch];
    s.total = n_layers * Hkv * s.tiles_sum;
    s.n_ctas = n_ctas; s.W = W;
    return s;
}

struct TilePos { int l, b, h, t, tiles_b, pair, pair_start; };

__device__ __forceinline__ TilePos locate(int x, const Sched &s, const int *pre)
{
    TilePos p;
    const int per_layer = s.Hkv * s.tiles_sum;
    p.l = x / per_layer;
    const int r = x - p.l * per_layer;
    int b = 0;
    while (b + 1 < s.batch && r >= pre[b + 1] * s.Hkv) ++b;
    p.b = b;
    p.tiles_b = pre[b + 1] - pre[b];
    const int r2 = r - pre[b] * s.Hkv;
    p.h = r2 / p.tiles_b;
    p.t = r2 - p.h * p.tiles_b;
    p.pair = (p.l * s.batch + b) * s.Hkv + p.h;
    p.pair_start = x - p.t;
    return p;
}


// host-side launchers of kernels that live in bgtq_decode.cu, for the other translation units
int launch_combine(const float *partials, const int32_t *seq_len, const float *rot128, int n_layers, int batch, int Hkv, int G,
                   int64_t n_cap, int n_ctas, int W, void *out, int n_sink, int n_recent, int win_slot, bool pdl, cudaStream_t st,
                   const HeadMeta *metas = nullptr, const float *rot_base = nullptr);   // metas: heads with V-side groups
int launch_window(const void *win_k, const void *win_v, const void *q, const int32_t *seq_len, const float *rot128_t,
                  float *partials, int pairs, int batch, int Hkv, int G, int64_t n_cap, int n_sink, int n_recent,
                  float scale_log2e, int win_slot, cudaStream_t st, const HeadMeta *metas = nullptr, const float *rot_t_base = nullptr,
                  bool pdl = false);   // pdl: programmatic launch (the kernel waits before it writes its record)
// bgtq_profile_decode: event pair around the split-KV kernel of a decode call (no-ops unless enabled)
bool profile_decode_on();
int profile_decode_begin(cudaStream_t st);
int profile_decode_end(cudaStream_t st);

}  // namespace bgtq
