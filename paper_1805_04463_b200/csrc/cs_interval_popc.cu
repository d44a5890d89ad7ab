// cs_interval_popc.cu -- stage a2, bit route: interval abundances by AND + POPC.
//
// Restates the paper's Alg. 20 (inner product of rows i and j between columns
// i and j, Fig. 4.2 caption PAPER.md:1768) for the GPU.  With bits = "future of i" (bits only at
// k > i) and bitsT = "past of j" (bits only at k < j), the word-wise AND is already restricted to
// i < k < j, so the paper's edge masks (Alg. 8) are not needed.
//
// Tiling: a persistent CTA takes 128 x 128 tiles (I <= J) of the pair space from a global counter,
// longest K range first.  For each tile it streams the rows future(i), i in tile I, and past(j),
// j in tile J, through shared memory in chunks of KC words with cp.async.bulk (one bulk copy per
// row per chunk, completion on an mbarrier), 2 stages.  Every thread keeps an 8 x 8 block of pair
// counters in registers: 16 shared-memory loads feed 64 AND+POPC per word.  The epilogue tests the
// relation bit of each pair and updates a shared-memory histogram (bins < HS; global atomics for
// the rare larger intervals), flushed to the int64 histogram with few global atomics.
#include <mutex>

#include "cs_common.cuh"

namespace cs {

namespace {

constexpr int TI = 128, TJ = 128;   // tile: rows i x rows j
constexpr int KC = 16;              // uint64 words per row per chunk (128 bytes)
constexpr int PITCH = KC * 8 + 16;  // bytes between rows in shared memory (bank spreading)
constexpr int NSTAGE = 2;
constexpr int HS = 2048;            // shared-memory histogram bins
constexpr int THREADS = 256;

constexpr int STAGE_BYTES = (TI + TJ) * PITCH;
constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + HS * 4 + 64;

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

struct TileCoord {
    int I, J;
};
// tiles ordered by decreasing K range: diagonal distance d = J - I from nT-1 down to 0
__device__ __forceinline__ TileCoord tile_from_index(int64_t t, int nT)
{
    int64_t m = (int64_t)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((m + 1) * (m + 2) / 2 <= t) m++;
    while (m * (m + 1) / 2 > t) m--;
    const int r = (int)(t - m * (m + 1) / 2);
    const int d = nT - 1 - (int)m;
    return TileCoord{r, r + d};
}

__global__ void __launch_bounds__(THREADS, 2)
k_interval_popc(const uint64_t *__restrict__ bits, const uint64_t *__restrict__ bitsT,
                int64_t B, int64_t N, int64_t stride, int64_t kmax,
                int64_t row_begin, int64_t row_end,
                unsigned long long *__restrict__ hist, unsigned long long *__restrict__ nrel,
                unsigned long long *tile_counter)
{
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *s_stage = smem;
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(smem + NSTAGE * STAGE_BYTES);
    uint64_t *s_bar = reinterpret_cast<uint64_t *>(smem + NSTAGE * STAGE_BYTES + HS * 4);
    long long *s_tile = reinterpret_cast<long long *>(s_bar + NSTAGE);
    unsigned long long *s_nrel = reinterpret_cast<unsigned long long *>(s_tile + 1);

    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const int nT = (int)((N + TI - 1) / TI);
    const int64_t tiles_per = (int64_t)nT * (nT + 1) / 2;
    const int64_t total_tiles = tiles_per * B;
    const int hs = (int)((kmax + 1 < HS) ? (kmax + 1) : HS);
    const int64_t hist_len = kmax + 1;

    if (tid == 0) {
        for (int s = 0; s < NSTAGE; s++) mbar_init(&s_bar[s], 1);
        *s_nrel = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int b = tid; b < HS; b += THREADS) s_hist[b] = 0;
    __syncthreads();

    uint32_t chunk_seq = 0;   // chunks issued so far by this CTA (stage = seq % NSTAGE, parity = seq / NSTAGE & 1)
    unsigned long long my_nrel = 0;
    int64_t cur_batch = -1;

    for (;;) {
        if (tid == 0) *s_tile = (long long)atomicAdd(tile_counter, 1ULL);
        __syncthreads();
        const int64_t t = *s_tile;
        __syncthreads();
        if (t >= total_tiles) break;
        const int64_t bidx = t / tiles_per;
        const TileCoord tc = tile_from_index(t - bidx * tiles_per, nT);
        const int64_t i0 = (int64_t)tc.I * TI, j0 = (int64_t)tc.J * TJ;
        if (i0 >= row_end || i0 + TI <= row_begin) continue;

        if (B > 1 && bidx != cur_batch) {   // per-causet histograms: flush before switching causet
            if (cur_batch >= 0) {
                for (int b = tid; b < hs; b += THREADS) {
                    uint32_t v = s_hist[b];
                    if (v) { atomicAdd(&hist[cur_batch * hist_len + b], (unsigned long long)v); s_hist[b] = 0; }
                }
                __syncthreads();
            }
            cur_batch = bidx;
        }
        if (B == 1) cur_batch = 0;

        const uint64_t *U = bits + bidx * N * stride;
        const uint64_t *L = bitsT + bidx * N * stride;
        const int vi = (int)((N - i0 < TI) ? (N - i0) : TI);   // valid rows in the tile
        const int vj = (int)((N - j0 < TJ) ? (N - j0) : TJ);
        const int64_t kbeg = i0 >> 6;                                     // first word that can hold k > i
        int64_t kend = ((j0 + TJ - 1) >> 6) + 1;                          // one past the last word with k < j
        if (kend > stride) kend = stride;
        const int nchunks = (int)((kend - kbeg + KC - 1) / KC);

        uint32_t acc[8][8];
#pragma unroll
        for (int a = 0; a < 8; a++)
#pragma unroll
            for (int c = 0; c < 8; c++) acc[a][c] = 0;

        auto issue = [&](int c, uint32_t seq) {
            const int s = seq % NSTAGE;
            const int64_t k0 = kbeg + (int64_t)c * KC;
            const int kw = (int)((kend - k0 < KC) ? (kend - k0) : KC);
            unsigned char *dstU = s_stage + s * STAGE_BYTES;
            unsigned char *dstL = dstU + TI * PITCH;
            if (tid == 0) mbar_arrive_expect_tx(&s_bar[s], (uint32_t)((vi + vj) * kw * 8));
            if (tid < TI) {
                if (tid < vi) bulk_g2s(dstU + tid * PITCH, U + (i0 + tid) * stride + k0, (uint32_t)(kw * 8), &s_bar[s]);
            } else {
                const int r = tid - TI;
                if (r < vj) bulk_g2s(dstL + r * PITCH, L + (j0 + r) * stride + k0, (uint32_t)(kw * 8), &s_bar[s]);
            }
        };

        issue(0, chunk_seq);
        for (int c = 0; c < nchunks; c++) {
            const uint32_t seq = chunk_seq + c;
            if (c + 1 < nchunks) issue(c + 1, seq + 1);
            const int s = seq % NSTAGE;
            mbar_wait(&s_bar[s], (seq / NSTAGE) & 1);
            const int64_t k0 = kbeg + (int64_t)c * KC;
            const int kw = (int)((kend - k0 < KC) ? (kend - k0) : KC);
            const unsigned char *pU = s_stage + s * STAGE_BYTES + ty * PITCH;
            const unsigned char *pL = s_stage + s * STAGE_BYTES + TI * PITCH + tx * PITCH;
#pragma unroll 2
            for (int k = 0; k < kw; k++) {
                uint64_t u[8], l[8];
#pragma unroll
                for (int a = 0; a < 8; a++) u[a] = *reinterpret_cast<const uint64_t *>(pU + a * 16 * PITCH + k * 8);
#pragma unroll
                for (int a = 0; a < 8; a++) l[a] = *reinterpret_cast<const uint64_t *>(pL + a * 16 * PITCH + k * 8);
#pragma unroll
                for (int a = 0; a < 8; a++)
#pragma unroll
                    for (int c2 = 0; c2 < 8; c2++) acc[a][c2] += __popcll(u[a] & l[c2]);
            }
            __syncthreads();   // everyone is done with stage s before it is refilled
        }
        chunk_seq += nchunks;

        // epilogue: relation bit of each pair, histogram update
#pragma unroll
        for (int a = 0; a < 8; a++) {
            const int64_t i = i0 + ty + 16 * a;
            if (i >= N || i < row_begin || i >= row_end) continue;
            const uint64_t r0 = U[i * stride + (j0 >> 6)];
            const uint64_t r1 = ((j0 >> 6) + 1 < stride) ? U[i * stride + (j0 >> 6) + 1] : 0ULL;
#pragma unroll
            for (int c2 = 0; c2 < 8; c2++) {
                const int jl = tx + 16 * c2;
                const uint64_t w = (jl < 64) ? r0 : r1;
                if ((w >> (jl & 63)) & 1ULL) {
                    my_nrel++;
                    const uint32_t cnt = acc[a][c2];
                    if (cnt < (uint32_t)hs) atomicAdd(&s_hist[cnt], 1u);
                    else if ((int64_t)cnt <= kmax) atomicAdd(&hist[cur_batch * hist_len + cnt], 1ULL);
                }
            }
        }
    }

    __syncthreads();
    if (cur_batch >= 0) {
        for (int b = tid; b < hs; b += THREADS) {
            uint32_t v = s_hist[b];
            if (v) atomicAdd(&hist[cur_batch * hist_len + b], (unsigned long long)v);
        }
    }
    if (nrel) {
        if (B == 1) {
#pragma unroll
            for (int s = 16; s >= 1; s >>= 1) my_nrel += __shfl_xor_sync(0xffffffffu, my_nrel, s);
            if ((tid & 31) == 0 && my_nrel) atomicAdd(s_nrel, my_nrel);
            __syncthreads();
            if (tid == 0 && *s_nrel) atomicAdd(nrel, *s_nrel);
        }
    }
}

}  // namespace

size_t interval_popc_scratch_bytes() { return 256; }

int launch_interval_popc(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                         int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                         void *scratch, cudaStream_t st)
{
    static PerDeviceFlag attr_set;
    const int dev = current_device();
    if (!attr_set.get(dev)) {
        CS_CUDA(cudaFuncSetAttribute(k_interval_popc, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
        attr_set.set(dev);
    }
    const int64_t stride = row_stride_words(N);
    // scratch = the workspace's IntervalStats block, zeroed by the caller; sched[0] is the tile counter
    const int64_t nT = (N + TI - 1) / TI;
    const int64_t total = nT * (nT + 1) / 2 * B;
    int64_t grid = (int64_t)sm_count() * 2;
    if (grid > total) grid = total;
    if (grid < 1) grid = 1;
    k_interval_popc<<<(unsigned)grid, THREADS, SMEM_BYTES, st>>>(
        bits, bitsT, B, N, stride, kmax, row_begin, row_end,
        reinterpret_cast<unsigned long long *>(hist), reinterpret_cast<unsigned long long *>(nrel),
        reinterpret_cast<unsigned long long *>(scratch));
    CS_LAUNCHED("k_interval_popc");
    return CS_OK;
}

// ---- a2 for callers that must not allocate: scratch in a static device array --------------------------------
// Some users of this library cannot hand over a workspace because they have no way to get one: code running inside
// another framework's allocator callback or with its caching allocator locked, a real-time or embedded service whose
// memory budget is fixed at start-up and forbids cudaMalloc afterwards, a plugin that is only given its input and
// output buffers.  For them the scratch of the bit route (the tile counter of k_interval_popc and, when the caller has
// no transposed matrix, the transposed matrix itself) lives in the array below, which is part of the library's device
// image: every GPU that loads libcausalset.so holds these 8 MiB + 256 B until the process exits.
//
// `g_static_scratch` is a device symbol.  In host code the name is only a stand-in the runtime uses to look the symbol
// up; it is NOT a device address, so it is never passed to a kernel or a memset.  static_scratch_address() asks the
// runtime for the real address once per device (with that device current) and caches it.
constexpr int64_t STATIC_MAX_N = 8192;
constexpr size_t STATIC_HEAD_BYTES = 256;                                  // IntervalStats block: sched[0] = tile counter
constexpr size_t STATIC_MAT_BYTES = (size_t)STATIC_MAX_N * (STATIC_MAX_N / 64) * 8;   // transposed matrix at the largest N
constexpr size_t STATIC_SCRATCH_BYTES = STATIC_HEAD_BYTES + STATIC_MAT_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

int64_t interval_static_max_n() { return STATIC_MAX_N; }

static int static_scratch_address(unsigned char **out)
{
    static unsigned char *addr[MAX_DEVICES];
    static std::mutex mu;
    int dev = -1;
    CS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cs_interval_hist_static: device ordinal %d is beyond the %d this library tracks",
                 dev, MAX_DEVICES);
        return CS_ERR_ARG;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void *p = nullptr;
        CS_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));   // the copy of the array that lives on the current device
        if (!p || ((uintptr_t)p & 255)) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "cs_interval_hist_static: bad address %p for the static scratch", p);
            return CS_ERR_CUDA;
        }
        CS_CUDA(cudaFuncSetAttribute(k_interval_popc, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
        addr[dev] = static_cast<unsigned char *>(p);
    }
    *out = addr[dev];
    return CS_OK;
}

// The same kernels as cs_interval_hist_ex(route = CS_ROUTE_POPC) on the whole row range; only where the scratch comes
// from differs.  No cudaMalloc / cudaFree / pool call on this path: memsets and launches only.
int launch_interval_popc_static(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                                int64_t *hist, int64_t *nrel, cudaStream_t st)
{
    if (N > STATIC_MAX_N) {
        snprintf(g_cuda_err, sizeof(g_cuda_err),
                 "cs_interval_hist_static: N = %lld is beyond the fixed capacity of the static scratch (N <= %lld); "
                 "use cs_interval_hist with a workspace", (long long)N, (long long)STATIC_MAX_N);
        return CS_ERR_CAPACITY;
    }
    kmax = clamp_kmax(N, kmax);
    CS_CUDA(cudaMemsetAsync(hist, 0, (size_t)(kmax + 1) * sizeof(int64_t), st));
    if (nrel) CS_CUDA(cudaMemsetAsync(nrel, 0, sizeof(int64_t), st));
    if (N < 2) return CS_OK;
    unsigned char *scratch = nullptr;
    int rc = static_scratch_address(&scratch);
    if (rc) return rc;
    // the array keeps what the last call left in it: the tile counter must start at zero; the transposed matrix is
    // overwritten whole (padding included) by launch_transpose_bits before the kernel reads it
    CS_CUDA(cudaMemsetAsync(scratch, 0, STATIC_HEAD_BYTES, st));
    if (!bitsT) {
        uint64_t *t = reinterpret_cast<uint64_t *>(scratch + STATIC_HEAD_BYTES);
        rc = launch_transpose_bits(bits, 1, N, t, st);
        if (rc) return rc;
        bitsT = t;
    }
    const int64_t stride = row_stride_words(N);
    const int64_t nT = (N + TI - 1) / TI;
    const int64_t total = nT * (nT + 1) / 2;
    int64_t grid = (int64_t)sm_count() * 2;
    if (grid > total) grid = total;
    k_interval_popc<<<(unsigned)grid, THREADS, SMEM_BYTES, st>>>(
        bits, bitsT, 1, N, stride, kmax, 0, N,
        reinterpret_cast<unsigned long long *>(hist), reinterpret_cast<unsigned long long *>(nrel),
        reinterpret_cast<unsigned long long *>(scratch));
    CS_LAUNCHED("k_interval_popc(static scratch)");
    return CS_OK;
}

}  // namespace cs
