// cs_peaks.cu -- peak probes: the measured denominators of bench.py's rooflines (cs_peak_probe).
//
// Not part of the path a1 -> a2 -> a3.  Each probe saturates ONE unit with the instruction the path's kernels
// use on it and reports units per second (CUDA events around the launch) and units per clock per SM (clock64
// inside the kernel), so that "fraction of the pipe's rate" in DESIGN.md / bench.py rests on a number measured
// on this pool's B200s instead of a nominal figure:
//   MXF4_PAIR  tcgen05.mma.cta_group::2.kind::mxf4.block_scale M=256 N=256 K=64, A in TMEM, B in shared memory
//              (the MMA of k_interval_pair), back to back on all CTA pairs
//   I8         tcgen05.mma.cta_group::1.kind::i8 M=128 N=256 K=32, A and B in shared memory (k_interval_tensor)
//   POPC       POPC.32 (k_interval_popc)           DFMA   fp64 fused multiply-add (the fp64 predicate of a1)
//   FFMA       fp32 FFMA                            FFMA2  fma.rn.f32x2 (the packed prefilter of a1)
//   HBM_WRITE  128-bit stores over the workspace    HBM_COPY  128-bit loads + stores
//   TMEM_LD    tcgen05.ld 32x32b.x32 from 4 or 8 warps of a CTA (the epilogue's accumulator drain)
//   MXF4_PAIR_N128  the MXF4_PAIR instruction with N = 128, alternating between two accumulator halves
//   MXF4_PAIR_N128_DEP  the same, every MMA accumulating into the same half (a dependent chain)
#include <vector>

#include "cs_common.cuh"

namespace cs {

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LAB_DONE;\n"
        "bra LAB_WAIT;\n"
        "LAB_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ bool elect_one()
{
    uint32_t p;
    asm volatile(
        "{\n"
        ".reg .pred q;\n"
        "elect.sync _|q, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, q;\n"
        "}\n"
        : "=r"(p));
    return p != 0;
}
// no swizzle, K-major; addresses and offsets in 16-byte units
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
__device__ __forceinline__ void tmem_st16_const(uint32_t taddr, uint32_t val)
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};\n" ::"r"(taddr),
        "r"(val)
        : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

constexpr int MMA_GROUP = 32;          // MMAs between two commits; two groups are in flight at most

// ---- kind::mxf4 on CTA pairs ----------------------------------------------------------------------
__host__ __device__ constexpr uint32_t mxf4_idesc(int n)
{
    return (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | (1u << 23) | ((uint32_t)(256 >> 4) << 24);
}

// NCOLS = 256: the MMA of k_interval_pair.  NCOLS = 128: the same with half the columns, alternating between two
// accumulator halves (independent chains) -- the shape a split accumulator would need.
template <int NCOLS, bool ALTERNATE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(128, 1)
k_probe_mxf4_pair(int groups, unsigned long long *__restrict__ clk)
{
    constexpr uint32_t MXF4_IDESC = mxf4_idesc(NCOLS);
    __shared__ __align__(1024) unsigned char s_b[4096];   // this CTA's half of B: 128 rows x K = 64 E2M1
    __shared__ uint64_t s_bar[2];
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t rank = cluster_ctarank();
    for (int i = tid; i < 1024; i += 128) reinterpret_cast<uint32_t *>(s_b)[i] = 0x22222222u;   // every element 1.0
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&s_tmem)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    const uint32_t lane_base = tmem + ((uint32_t)(warp * 32) << 16);
    tmem_st16_const(lane_base + 256, 0x7F7F7F7Fu);    // unit UE8M0 scales
    tmem_st16_const(lane_base + 320, 0x22222222u);    // A: 128 rows x K = 64 (8 columns) of 1.0, and spare
    tc_fence_before();
    __syncthreads();
    cluster_sync();
    tc_fence_after();
    if (warp == 0 && rank == 0) {
        const uint64_t bd = make_desc(smem_u32(s_b), (NCOLS / 2) * 16, 128);
        unsigned long long t0 = 0;
        for (int g = 0; g < groups; g++) {
            if (g >= 2) mbar_wait(&s_bar[g & 1], ((g >> 1) - 1) & 1);     // group g-2 has retired
            if (g == 2) t0 = clock64();                                   // the pipe is full from here on
            if (elect_one()) {
#pragma unroll 4
                for (int i = 0; i < MMA_GROUP; i++) {
                    const uint32_t d = tmem + (ALTERNATE ? (uint32_t)(i & 1) * 128u : 0u);
                    asm volatile(
                        "{\n"
                        ".reg .pred p;\n"
                        "setp.ne.b32 p, %4, 0;\n"
                        "tcgen05.mma.cta_group::2.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%5], [%5], p;\n"
                        "}\n" ::"r"(d),
                        "r"(tmem + 320), "l"(bd), "r"(MXF4_IDESC), "r"((uint32_t)((g | (i >> 1)) != 0)), "r"(tmem + 256)
                        : "memory");
                }
                asm volatile(
                    "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                        smem_u32(&s_bar[g & 1])),
                    "h"((uint16_t)1)
                    : "memory");
            }
            __syncwarp();
        }
        // groups g = groups-2 and groups-1 are still in flight
        if (groups >= 2) mbar_wait(&s_bar[groups & 1], ((groups >> 1) - 1) & 1);
        if (groups >= 1) mbar_wait(&s_bar[(groups - 1) & 1], ((groups - 1) >> 1) & 1);
        const unsigned long long t1 = clock64();
        if (tid == 0) clk[blockIdx.x >> 1] = t1 - t0;      // covers groups 2 .. groups-1 (plus the drain of two)
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

// ---- kind::i8, one CTA ------------------------------------------------------------------------------
constexpr uint32_t I8_IDESC = (2u << 4) | ((uint32_t)(256 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

__global__ void __launch_bounds__(128, 1) k_probe_i8(int groups, unsigned long long *__restrict__ clk)
{
    __shared__ __align__(1024) unsigned char s_a[4096];   // 128 rows x K = 32 bytes
    __shared__ __align__(1024) unsigned char s_b[8192];   // 256 rows x K = 32 bytes
    __shared__ uint64_t s_bar[2];
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 1024; i += 128) reinterpret_cast<uint32_t *>(s_a)[i] = 0x01010101u;
    for (int i = tid; i < 2048; i += 128) reinterpret_cast<uint32_t *>(s_b)[i] = 0x01010101u;
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&s_tmem)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    if (warp == 0) {
        const uint64_t ad = make_desc(smem_u32(s_a), 128 * 16, 128);
        const uint64_t bd = make_desc(smem_u32(s_b), 256 * 16, 128);
        unsigned long long t0 = 0;
        for (int g = 0; g < groups; g++) {
            if (g >= 2) mbar_wait(&s_bar[g & 1], ((g >> 1) - 1) & 1);
            if (g == 2) t0 = clock64();
            if (elect_one()) {
#pragma unroll 4
                for (int i = 0; i < MMA_GROUP; i++) {
                    asm volatile(
                        "{\n"
                        ".reg .pred p;\n"
                        "setp.ne.b32 p, %4, 0;\n"
                        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n"
                        "}\n" ::"r"(tmem),
                        "l"(ad), "l"(bd), "r"(I8_IDESC), "r"((uint32_t)(i != 0))
                        : "memory");
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                                 smem_u32(&s_bar[g & 1]))
                             : "memory");
            }
            __syncwarp();
        }
        if (groups >= 2) mbar_wait(&s_bar[groups & 1], ((groups >> 1) - 1) & 1);
        if (groups >= 1) mbar_wait(&s_bar[(groups - 1) & 1], ((groups - 1) >> 1) & 1);
        const unsigned long long t1 = clock64();
        if (tid == 0) clk[blockIdx.x] = t1 - t0;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

// ---- tcgen05.ld ---------------------------------------------------------------------------------------
// WARPS warps (4: one per TMEM lane quarter; 8: two per quarter, as in k_interval_pair's epilogue) read
// 32 lanes x 128 columns per iteration.  4096 bytes per instruction and warp.
__global__ void __launch_bounds__(256, 1) k_probe_tmem_ld(int iters, int warps, unsigned long long *__restrict__ clk,
                                                          uint32_t *__restrict__ sink)
{
    __shared__ uint32_t s_tmem;
    __shared__ unsigned long long s_max;
    const int tid = threadIdx.x, warp = tid >> 5;
    if (tid == 0) s_max = 0;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&s_tmem)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    if (warp < warps) {
        const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (warp >> 2) * 128;
        uint32_t acc = 0;
        const unsigned long long t0 = clock64();
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int c = 0; c < 4; c++) {
                uint32_t v[32];
                asm volatile(
                    "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                    "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                    "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
                    : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                      "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
                      "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]),
                      "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]),
                      "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                    : "r"(taddr + c * 32)
                    : "memory");
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                acc ^= v[0] ^ v[13] ^ v[31];
            }
        }
        const unsigned long long t1 = clock64();
        if (acc == 0x9e3779b9u) sink[0] = acc;      // keeps the loads alive
        if ((tid & 31) == 0) atomicMax(&s_max, t1 - t0);
    }
    tc_fence_before();
    __syncthreads();
    if (tid == 0) clk[blockIdx.x] = s_max;
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

// ---- SIMT pipes -----------------------------------------------------------------------------------------
enum { ALU_POPC = 0, ALU_DFMA = 1, ALU_FFMA = 2, ALU_FFMA2 = 3 };
constexpr int CHAINS = 8, ALU_UNROLL = 16;

template <int WHICH>
__global__ void __launch_bounds__(512, 2) k_probe_alu(int iters, unsigned long long *__restrict__ clk, uint32_t *__restrict__ sink)
{
    __shared__ unsigned long long s_max;
    if (threadIdx.x == 0) s_max = 0;
    __syncthreads();
    const uint32_t seed = threadIdx.x * 2654435761u + blockIdx.x;
    unsigned long long t0, t1;
    uint32_t out = 0;
    if (WHICH == ALU_POPC) {
        uint32_t x[CHAINS];
#pragma unroll
        for (int c = 0; c < CHAINS; c++) x[c] = seed + c;
        t0 = clock64();
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int u = 0; u < ALU_UNROLL; u++)
#pragma unroll
                for (int c = 0; c < CHAINS; c++) x[c] = __popc(x[c]) + seed;     // POPC feeds an IADD: a dependent chain
        }
        t1 = clock64();
#pragma unroll
        for (int c = 0; c < CHAINS; c++) out ^= x[c];
    } else if (WHICH == ALU_DFMA) {
        double x[CHAINS];
        const double a = 1.0 + (double)(seed & 7) * 1e-9, b = 1e-9;
#pragma unroll
        for (int c = 0; c < CHAINS; c++) x[c] = (double)c;
        t0 = clock64();
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int u = 0; u < ALU_UNROLL; u++)
#pragma unroll
                for (int c = 0; c < CHAINS; c++) x[c] = fma(x[c], a, b);
        }
        t1 = clock64();
#pragma unroll
        for (int c = 0; c < CHAINS; c++) out ^= (uint32_t)__double2hiint(x[c]);
    } else if (WHICH == ALU_FFMA) {
        float x[CHAINS];
        const float a = 1.0f + (float)(seed & 7) * 1e-6f, b = 1e-6f;
#pragma unroll
        for (int c = 0; c < CHAINS; c++) x[c] = (float)c;
        t0 = clock64();
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int u = 0; u < ALU_UNROLL; u++)
#pragma unroll
                for (int c = 0; c < CHAINS; c++) x[c] = fmaf(x[c], a, b);
        }
        t1 = clock64();
#pragma unroll
        for (int c = 0; c < CHAINS; c++) out ^= __float_as_uint(x[c]);
    } else {
        unsigned long long x[CHAINS];
        const float af = 1.0f + (float)(seed & 7) * 1e-6f;
        const unsigned long long a = ((unsigned long long)__float_as_uint(af) << 32) | __float_as_uint(af);
        const unsigned long long b = ((unsigned long long)__float_as_uint(1e-6f) << 32) | __float_as_uint(2e-6f);
#pragma unroll
        for (int c = 0; c < CHAINS; c++) x[c] = (unsigned long long)__float_as_uint((float)c) * 0x100000001ull;
        t0 = clock64();
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int u = 0; u < ALU_UNROLL; u++)
#pragma unroll
                for (int c = 0; c < CHAINS; c++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[c]) : "l"(a), "l"(b));
        }
        t1 = clock64();
#pragma unroll
        for (int c = 0; c < CHAINS; c++) out ^= (uint32_t)x[c] ^ (uint32_t)(x[c] >> 32);
    }
    if (out == 0x12345u) sink[1] = out;
    if ((threadIdx.x & 31) == 0) atomicMax(&s_max, t1 - t0);
    __syncthreads();
    if (threadIdx.x == 0) clk[blockIdx.x] = s_max;
}

// ---- HBM ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_hbm_write(uint4 *__restrict__ dst, size_t n16)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const uint4 v = make_uint4(blockIdx.x, threadIdx.x, 3u, 4u);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) dst[i] = v;
}
__global__ void __launch_bounds__(256) k_probe_hbm_copy(const uint4 *__restrict__ src, uint4 *__restrict__ dst, size_t n16)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) dst[i] = src[i];
}

}  // namespace

// out_host: {units, seconds, units per clock per SM (0 where clocks are not taken)}
int launch_peak_probe(int kind, int64_t iters, void *workspace, size_t workspace_bytes, double *out_host, cudaStream_t st)
{
    if (!workspace || workspace_bytes < 65536 || ((uintptr_t)workspace & 255)) return CS_ERR_WORKSPACE;
    if (iters < 4) iters = 4;
    if (iters > (1 << 22)) iters = 1 << 22;
    const int sms = sm_count();
    unsigned long long *clk = static_cast<unsigned long long *>(workspace);           // [<= 4096]
    uint32_t *sink = reinterpret_cast<uint32_t *>(static_cast<unsigned char *>(workspace) + 32768);
    CS_CUDA(cudaMemsetAsync(workspace, 0, 65536, st));
    cudaEvent_t e0, e1;
    CS_CUDA(cudaEventCreate(&e0));
    if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return cuda_fail(cudaGetLastError(), "cudaEventCreate"); }
    double units = 0.0, per_clk_units = 0.0;   // per_clk_units: units one clock-reporting CTA (or pair) executed
    int nclk = 0, sms_per_clk = 1;
    int rc = CS_OK;
    auto launch = [&]() -> int {
        switch (kind) {
        case CS_PEAK_MXF4_PAIR:
        case CS_PEAK_MXF4_PAIR_N128:
        case CS_PEAK_MXF4_PAIR_N128_DEP: {
            const int groups = (int)((iters + MMA_GROUP - 1) / MMA_GROUP) + 2;
            const double ncols = kind == CS_PEAK_MXF4_PAIR ? 256.0 : 128.0;
            if (kind == CS_PEAK_MXF4_PAIR) k_probe_mxf4_pair<256, false><<<sms / 2 * 2, 128, 0, st>>>(groups, clk);
            else if (kind == CS_PEAK_MXF4_PAIR_N128) k_probe_mxf4_pair<128, true><<<sms / 2 * 2, 128, 0, st>>>(groups, clk);
            else k_probe_mxf4_pair<128, false><<<sms / 2 * 2, 128, 0, st>>>(groups, clk);
            units = 2.0 * 256 * ncols * 64 * MMA_GROUP * (double)groups * (sms / 2);
            per_clk_units = 2.0 * 256 * ncols * 64 * MMA_GROUP * (double)(groups - 2);
            nclk = sms / 2; sms_per_clk = 2;
            break;
        }
        case CS_PEAK_I8: {
            const int groups = (int)((iters + MMA_GROUP - 1) / MMA_GROUP) + 2;
            k_probe_i8<<<sms, 128, 0, st>>>(groups, clk);
            units = 2.0 * 128 * 256 * 32 * MMA_GROUP * (double)groups * sms;
            per_clk_units = 2.0 * 128 * 256 * 32 * MMA_GROUP * (double)(groups - 2);
            nclk = sms;
            break;
        }
        case CS_PEAK_TMEM_LD4:
        case CS_PEAK_TMEM_LD8: {
            const int warps = kind == CS_PEAK_TMEM_LD4 ? 4 : 8;
            k_probe_tmem_ld<<<sms, 256, 0, st>>>((int)iters, warps, clk, sink);
            per_clk_units = 4.0 * 4096 * (double)iters * warps;   // bytes per CTA
            units = per_clk_units * sms;
            nclk = sms;
            break;
        }
        case CS_PEAK_POPC:
        case CS_PEAK_DFMA:
        case CS_PEAK_FFMA:
        case CS_PEAK_FFMA2: {
            const int ctas = 2 * sms;
            if (kind == CS_PEAK_POPC) k_probe_alu<ALU_POPC><<<ctas, 512, 0, st>>>((int)iters, clk, sink);
            else if (kind == CS_PEAK_DFMA) k_probe_alu<ALU_DFMA><<<ctas, 512, 0, st>>>((int)iters, clk, sink);
            else if (kind == CS_PEAK_FFMA) k_probe_alu<ALU_FFMA><<<ctas, 512, 0, st>>>((int)iters, clk, sink);
            else k_probe_alu<ALU_FFMA2><<<ctas, 512, 0, st>>>((int)iters, clk, sink);
            // lane-operations: one POPC.32 / DFMA / FFMA per lane; FFMA2 counts two fused multiply-adds per lane
            per_clk_units = 512.0 * CHAINS * ALU_UNROLL * (double)iters * (kind == CS_PEAK_FFMA2 ? 2.0 : 1.0) * 2.0;   // two CTAs per SM
            units = per_clk_units * sms;
            nclk = ctas;
            break;
        }
        case CS_PEAK_HBM_WRITE:
        case CS_PEAK_HBM_COPY: {
            const size_t avail = (workspace_bytes - 65536) / 32 * 32;
            if (avail < ((size_t)1 << 28)) return CS_ERR_WORKSPACE;     // must dwarf the 126 MB L2
            uint4 *base = reinterpret_cast<uint4 *>(static_cast<unsigned char *>(workspace) + 65536);
            if (kind == CS_PEAK_HBM_WRITE) {
                k_probe_hbm_write<<<sms * 16, 256, 0, st>>>(base, avail / 16);
                units = (double)avail;
            } else {
                k_probe_hbm_copy<<<sms * 16, 256, 0, st>>>(base, base + avail / 32, avail / 32);
                units = (double)avail;          // half read + half written
            }
            break;
        }
        default:
            return CS_ERR_ARG;
        }
        return CS_OK;
    };
    // one untimed pass (instruction cache, clocks), one timed
    for (int pass = 0; pass < 2 && rc == CS_OK; pass++) {
        if (pass == 1 && cudaEventRecord(e0, st) != cudaSuccess) rc = CS_ERR_CUDA;
        if (rc == CS_OK) rc = launch();
        if (rc == CS_OK) {
            g_launches++;
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) rc = cuda_fail(e, "peak probe launch");
        }
    }
    float ms = 0.f;
    if (rc == CS_OK) {
        cudaError_t e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) rc = cuda_fail(e, "peak probe timing");
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc != CS_OK) return rc;
    out_host[0] = units;
    out_host[1] = ms * 1e-3;
    out_host[2] = 0.0;
    if (nclk > 0) {
        if (nclk > 4096) return CS_ERR_ARG;
        std::vector<unsigned long long> h((size_t)nclk, 0ull);
        cudaError_t e = cudaMemcpy(h.data(), clk, (size_t)nclk * 8, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(e, "peak probe clocks");
        unsigned long long worst = 0;
        for (int i = 0; i < nclk; i++) worst = h[i] > worst ? h[i] : worst;
        if (worst) out_host[2] = per_clk_units / (double)worst / sms_per_clk;
    }
    return CS_OK;
}

}  // namespace cs
