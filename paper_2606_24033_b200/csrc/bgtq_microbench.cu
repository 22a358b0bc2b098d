// bgtq_microbench.cu -- the instruction-rate microbenchmarks the profile notes quote (bgtq_debug_microbench; used by
// `bench.py --microbench` and tests/test_gpu_microbench.py, never by the product path).  They answer three questions about
// one B200 SM that the design of the decode kernels hangs on:
//   1. which instructions share the half-rate "ALU" pipe (PRMT / LOP3 / SHF) and which do not (IMAD, HFMA2, FFMA, IADD);
//   2. what a 3-bit unit (1024 codes) costs to unpack to fp16 mma.sync fragments (round-1 decoder) and to e4m3 byte planes;
//   3. how fast ONE thread can issue tcgen05.mma (about one per 60 clocks, whatever N) and how that scales with issuers.
#include <cstdint>
#include <cstring>

#include "bgtq_internal.h"
#include "bgtq_device.cuh"

namespace bgtq {

#define CUDA_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_, #expr); } while (0)

// ---------------------------------------------------------------- 1. pipe mixes: 8 independent chains per thread
// MODE bits: 1 PRMT, 2 IMAD, 4 FFMA, 8 HFMA2, 16 LOP3 (3 register inputs), 32 SHF (funnel), 64 IADD, 128 FMNMX
template <int MODE>
__global__ void __launch_bounds__(512) mb_pipe_kernel(int iters, uint32_t *out, long long *cyc, uint32_t seed)
{
    uint32_t x[8], y[8], z[8];
    float f[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { x[i] = seed + threadIdx.x * 17 + i; y[i] = seed * 3 + i + threadIdx.x * 7; z[i] = y[i] ^ x[i]; f[i] = (float)(threadIdx.x + i); }
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE & 1) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(x[i]) : "r"(seed), "r"(0x3210u + i));
                if (MODE & 2) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(y[i]) : "r"(3u), "r"(seed));
                if (MODE & 4) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(1.0001f), "f"(0.5f));
                if (MODE & 8) asm volatile("fma.rn.f16x2 %0, %0, %1, %2;" : "+r"(z[i]) : "r"(0x3c003c00u), "r"(seed));
                if (MODE & 16) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(z[i]) : "r"(x[i]), "r"(x[(i + 1) & 7]));
                if (MODE & 32) asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(z[i]) : "r"(x[i]), "r"(x[(i + 1) & 7]));
                if (MODE & 64) asm volatile("add.u32 %0, %0, %1;" : "+r"(y[i]) : "r"(x[i]));
                if (MODE & 128) asm volatile("max.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(__uint_as_float(y[i])));
            }
    }
    const long long t1 = clock64();
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += x[i] + y[i] + z[i] + __float_as_uint(f[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// ---------------------------------------------------------------- 2. unpack loops from shared memory (3-bit units)
__device__ __forceinline__ void mb_dec3_f16(const uint32_t (&w)[3], const uint32_t *pools, uint32_t (&h)[16])
{
    const uint32_t LOa = pools[0], LOb = pools[1], HIa = pools[2], HIb = pools[3];
    uint32_t t[4];
    t[0] = w[0] & 0x77777777u; t[1] = w[1] & 0x77777777u; t[2] = w[2] & 0x77777777u;
    t[3] = ((w[0] >> 3) & 0x11111111u) | ((w[1] >> 2) & 0x22222222u) | ((w[2] >> 1) & 0x44444444u);
#pragma unroll
    for (int wi = 0; wi < 4; ++wi)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
            const uint32_t sel = hf ? (t[wi] >> 16) : t[wi];
            const uint32_t lo4 = prmt(LOa, LOb, sel), hi4 = prmt(HIa, HIb, sel);
            h[wi * 4 + 2 * hf] = prmt(lo4, hi4, 0x5140);
            h[wi * 4 + 2 * hf + 1] = prmt(lo4, hi4, 0x7362);
        }
}
__device__ __forceinline__ void mb_dec3_f8(const uint32_t (&w)[3], const uint32_t *pools, uint32_t (&hi)[8], uint32_t (&lo)[8])
{
    const uint32_t LOa = pools[0], LOb = pools[1], HIa = pools[2], HIb = pools[3];
    uint32_t t[4];
    t[0] = w[0] & 0x77777777u; t[1] = w[1] & 0x77777777u; t[2] = w[2] & 0x77777777u;
    t[3] = ((w[0] >> 3) & 0x11111111u) | ((w[1] >> 2) & 0x22222222u) | ((w[2] >> 1) & 0x44444444u);
#pragma unroll
    for (int wi = 0; wi < 4; ++wi)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
            const uint32_t sel = hf ? (t[wi] >> 16) : t[wi];
            lo[wi * 2 + hf] = prmt(LOa, LOb, sel);
            hi[wi * 2 + hf] = prmt(HIa, HIb, sel);
        }
}
__device__ __forceinline__ void mb_hmma(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mb_tf32(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// MODE 0: two units -> fp16 fragments + 8 HMMA (the round-1 PV loop body); 1: fp16 decode only; 2: e4m3 planes decode only;
// 3: 8 HMMA only (issue rate of the legacy tensor path); 4: 8 TF32 m16n8k8 MMAs only (the append fast path's rotation)
template <int MODE>
__global__ void __launch_bounds__(512) mb_unpack_kernel(int iters, int units, uint32_t *out, long long *cyc, const uint32_t *src)
{
    extern __shared__ uint32_t mb_sm[];
    __shared__ uint32_t pools[4];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    uint32_t *buf = mb_sm + warp * units * 96;
    for (int i = lane; i < units * 96; i += 32) buf[i] = src[(blockIdx.x * nw + warp) * 64 + (i & 63)] * 2654435761u + i;
    if (threadIdx.x < 4) pools[threadIdx.x] = src[threadIdx.x] | 0x01010101u;
    __syncthreads();
    float C[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i) C[i][0] = C[i][1] = C[i][2] = C[i][3] = 0.f;
    uint32_t fold = 0;
    const uint32_t b0 = src[lane], b1 = src[lane + 32];
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it)
#pragma unroll 1
        for (int u = 0; u < units; u += 2) {
            const uint32_t *p = buf + u * 96 + lane;
            uint32_t w0[3], w1[3];
#pragma unroll
            for (int i = 0; i < 3; ++i) { w0[i] = p[i * 32]; w1[i] = p[96 + i * 32]; }
            if (MODE == 0 || MODE == 1) {
                uint32_t h0[16], h1[16];
                mb_dec3_f16(w0, pools, h0);
                mb_dec3_f16(w1, pools, h1);
                if (MODE == 0) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) mb_hmma(C[i], h0[2 * i], h0[2 * i + 1], h1[2 * i], h1[2 * i + 1], b0, b1);
                } else {
#pragma unroll
                    for (int i = 0; i < 16; ++i) fold ^= h0[i] ^ h1[i];
                }
            } else if (MODE == 2) {
                uint32_t hi[8], lo[8];
                mb_dec3_f8(w0, pools, hi, lo);
#pragma unroll
                for (int i = 0; i < 8; ++i) fold ^= hi[i] ^ lo[i];
                mb_dec3_f8(w1, pools, hi, lo);
#pragma unroll
                for (int i = 0; i < 8; ++i) fold ^= hi[i] ^ lo[i];
            } else if (MODE == 4) {
#pragma unroll
                for (int i = 0; i < 8; ++i) mb_tf32(C[i], w0[0], w0[1], w0[2], w1[0], b0, b1);
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) mb_hmma(C[i], w0[0], w0[1], w0[2], w1[0], b0, b1);
            }
        }
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += C[i][0] + C[i][1] + C[i][2] + C[i][3];
    out[blockIdx.x * blockDim.x + threadIdx.x] = __float_as_uint(acc) ^ fold;
    __syncthreads();
    if (threadIdx.x == 0) cyc[blockIdx.x] = clock64() - t0;
}

// ---------------------------------------------------------------- 3. tcgen05.mma issue rate (M = 128, N = 8, K = 32 e4m3, A in tensor memory)
// NI warps each issue n_mma instructions from one thread into their own accumulator columns; time until all have completed.
template <int NI>
__global__ void __launch_bounds__(128) mb_umma_kernel(int n_mma, long long *cyc)
{
    extern __shared__ __align__(1024) uint8_t mb_raw[];
    uint8_t *sm = mb_raw + ((1024u - (smem_u32(mb_raw) & 1023u)) & 1023u);
    __shared__ uint32_t tmem_base_s;
    __shared__ __align__(8) uint64_t bar[4];
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 4096 / 4; i += 128) reinterpret_cast<uint32_t *>(sm)[i] = 0x38383838u;     // e4m3 1.0
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" :: "r"(smem_u32(&tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        for (int i = 0; i < 4; ++i) mbar_init(smem_u32(&bar[i]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tb = tmem_base_s;
    const long long t0 = clock64();
    if ((tid & 31) == 0 && warp < NI) {
        constexpr uint32_t idesc = (1u << 4) | (1u << 17) | (8u << 24);
        const uint64_t dbase = (uint64_t)((smem_u32(sm) & 0x3FFFF) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
                               ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
        for (int i = 0; i < n_mma; ++i) {
            const uint32_t d = tb + 256 + warp * 64 + (i & 7) * 8, a = tb + warp * 64 + (i & 7) * 8;
            const uint64_t db = dbase + (uint64_t)((i & 3) * 2);
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                         "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}"
                         :: "r"(d), "r"(a), "l"(db), "r"(idesc), "r"(1u) : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&bar[warp])) : "memory");
        mbar_wait(smem_u32(&bar[warp]), 0);
    }
    __syncthreads();
    if (tid == 0) cyc[blockIdx.x] = clock64() - t0;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tb) : "memory");
}

// ---------------------------------------------------------------- host dispatcher
static const char *const kMbNames[BGTQ_MICROBENCH_COUNT] = {
    "PRMT: warp-instructions per clock per scheduler",
    "LOP3 (3 registers)", "SHF (funnel)", "IMAD", "HFMA2", "FFMA", "IADD", "FMNMX",
    "PRMT + LOP3 (same pipe)", "PRMT + SHF (same pipe)", "PRMT + IMAD", "PRMT + HFMA2", "PRMT + FFMA", "PRMT + IMAD + FFMA",
    "HMMA.16816: clocks per instruction per scheduler",
    "3-bit unit -> fp16 fragments + HMMA: SM clocks per unit (1024 codes)",
    "3-bit unit -> fp16 fragments, decode only: SM clocks per unit",
    "3-bit unit -> e4m3 hi/lo byte planes, decode only: SM clocks per unit",
    "tcgen05.mma M128 N8 K32 (A in TMEM), 1 issuing thread: clocks per MMA",
    "tcgen05.mma, 2 issuing threads: clocks per MMA overall",
    "tcgen05.mma, 4 issuing threads: clocks per MMA overall",
    "HMMA.1688.TF32 (mma.sync m16n8k8 tf32): clocks per instruction per scheduler",
};

const char *microbench_name(int which) { return which >= 0 && which < BGTQ_MICROBENCH_COUNT ? kMbNames[which] : nullptr; }

template <typename F>
static int mb_time(F launch, int grid, double *mean_cycles)
{
    long long *d_cyc = nullptr;
    std::vector<long long> h(grid);
    CUDA_TRY(cudaMalloc(&d_cyc, grid * sizeof(long long)));
    launch(d_cyc, true);                                      // warm-up
    launch(d_cyc, false);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(h.data(), d_cyc, grid * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaFree(d_cyc);
    if (e != cudaSuccess) return cuda_fail(e, "bgtq_debug_microbench");
    double s = 0;
    for (long long v : h) s += (double)v;
    *mean_cycles = s / grid;
    return BGTQ_OK;
}

int microbench_run(int which, int warps, double *value)
{
    const int grid = 148, iters = 2000, W = warps;
    uint32_t *out = nullptr, *src = nullptr;
    CUDA_TRY(cudaMalloc(&out, grid * 512 * 4));
    CUDA_TRY(cudaMalloc(&src, 1 << 20));
    {
        std::vector<uint32_t> h(1 << 18);
        uint32_t s = 12345u;
        for (auto &v : h) { s = s * 1664525u + 1013904223u; v = s; }
        CUDA_TRY(cudaMemcpy(src, h.data(), 1 << 20, cudaMemcpyHostToDevice));
    }
    double c = 0;
    int rc = BGTQ_OK;
    auto pipe = [&](auto kern, int n_instr) {
        rc = mb_time([&](long long *cyc, bool warm) { kern<<<grid, W * 32>>>(warm ? 10 : iters, out, cyc, 12345u); count_launch(); }, grid, &c);
        *value = (double)iters * n_instr * W / 4.0 / c;
    };
    auto unpack = [&](auto kern, int units_per_iter_denominator) {
        const int units = 16, it2 = 200;
        const size_t smem = (size_t)W * units * 96 * 4;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        rc = mb_time([&](long long *cyc, bool warm) { kern<<<grid, W * 32, smem>>>(warm ? 2 : it2, units, out, cyc, src); count_launch(); }, grid, &c);
        *value = c / ((double)it2 * units * W) * units_per_iter_denominator;
    };
    auto umma = [&](auto kern, int ni) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 8 * 1024);
        rc = mb_time([&](long long *cyc, bool) { kern<<<grid, 128, 8 * 1024>>>(1000, cyc); count_launch(); }, grid, &c);
        *value = c / 1000.0 / ni;
    };
    switch (which) {
    case 0: pipe(mb_pipe_kernel<1>, 32); break;
    case 1: pipe(mb_pipe_kernel<16>, 32); break;
    case 2: pipe(mb_pipe_kernel<32>, 32); break;
    case 3: pipe(mb_pipe_kernel<2>, 32); break;
    case 4: pipe(mb_pipe_kernel<8>, 32); break;
    case 5: pipe(mb_pipe_kernel<4>, 32); break;
    case 6: pipe(mb_pipe_kernel<64>, 32); break;
    case 7: pipe(mb_pipe_kernel<128>, 32); break;
    case 8: pipe(mb_pipe_kernel<1 | 16>, 64); break;
    case 9: pipe(mb_pipe_kernel<1 | 32>, 64); break;
    case 10: pipe(mb_pipe_kernel<1 | 2>, 64); break;
    case 11: pipe(mb_pipe_kernel<1 | 8>, 64); break;
    case 12: pipe(mb_pipe_kernel<1 | 4>, 64); break;
    case 13: pipe(mb_pipe_kernel<1 | 2 | 4>, 96); break;
    case 14: unpack(mb_unpack_kernel<3>, 1); *value = *value * 2.0 * 4.0 / 8.0; break;   // SM clocks per 2 units -> per HMMA per scheduler
    case 15: unpack(mb_unpack_kernel<0>, 1); break;
    case 16: unpack(mb_unpack_kernel<1>, 1); break;
    case 17: unpack(mb_unpack_kernel<2>, 1); break;
    case 18: umma(mb_umma_kernel<1>, 1); break;
    case 19: umma(mb_umma_kernel<2>, 2); break;
    case 20: umma(mb_umma_kernel<4>, 4); break;
    case 21: unpack(mb_unpack_kernel<4>, 1); *value = *value * 2.0 * 4.0 / 8.0; break;
    default: rc = BGTQ_EINVAL; set_error("bgtq_debug_microbench: unknown benchmark"); break;
    }
    cudaFree(out);
    cudaFree(src);
    return rc;
}

}  // namespace bgtq
