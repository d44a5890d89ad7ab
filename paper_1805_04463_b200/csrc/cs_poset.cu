// cs_poset.cu -- NEXT-3: chain and antichain primitives on the bit matrix (Algorithms 11-13,
// PAPER.md:1265-1403).
//
// Longest chains (Algorithm 11 computes, by memoised recursion through the Alexandroff set, the
// longest chain between two elements).  Here every element gets its height at once: height[k] = number
// of elements of the longest chain ending at k = 1 + max over predecessors.  The recursion is
// sequential; the bit matrix allows peeling instead: level l is the set of remaining elements none of
// whose predecessors remain (past(k) & R == 0, one AND per 64 elements, scanned from k downwards
// because the predecessors that remain longest are the latest ones).  With a source element the
// remaining set starts as J+(source), which by transitivity contains every element of every chain from it.
//
// Greedy maximal antichain (Algorithm 13): per step c(j) = |A \ J(j)| for every candidate j is one
// AND-NOT + POPC sweep over the rows of bits | bitsT; the first j with the largest c wins
// (64-bit atomicMax of c << 32 | ~j), then A and the candidates lose J(k).
//
// Both are persistent cooperative kernels: the steps depend on each other, a grid-wide barrier separates them.
#include <cooperative_groups.h>

#include "cs_common.cuh"

namespace cg = cooperative_groups;

namespace cs {

namespace {

constexpr int POSET_THREADS = 256;

// state block in the workspace
struct PosetState {
    unsigned long long best[2];    // antichain: packed (c << 32 | ~j) of the step's winner, two slots alternate
    long long remaining;           // chains: elements not yet assigned
    long long longest;
};

__global__ void __launch_bounds__(POSET_THREADS)
k_chain_heights(const uint64_t *__restrict__ bits, const uint64_t *__restrict__ bitsT, int64_t N, int64_t stride,
                int64_t source, int32_t *__restrict__ height, uint64_t *R0, uint64_t *R1, PosetState *st,
                long long *longest_out)
{
    cg::grid_group grid = cg::this_grid();
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nthreads = (int64_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    const int64_t warp = tid >> 5, nwarps = nthreads >> 5;
    const int64_t words = (N + 63) >> 6;

    // initial remaining set and heights
    for (int64_t w = tid; w < stride; w += nthreads) {
        uint64_t r;
        if (source >= 0) r = bits[source * stride + w];                      // J+(source)
        else r = w < words ? ((w == words - 1 && (N & 63)) ? (~0ULL >> (64 - (N & 63))) : ~0ULL) : 0ULL;
        R0[w] = r;
    }
    for (int64_t k = tid; k < N; k += nthreads) height[k] = (k == source) ? 1 : 0;
    if (tid == 0) {
        st->remaining = 0;
        st->longest = (source >= 0) ? 1 : 0;
    }
    grid.sync();
    {   // count the remaining elements
        long long c = 0;
        for (int64_t w = tid; w < stride; w += nthreads) c += __popcll(R0[w]);
        for (int s = 16; s >= 1; s >>= 1) c += __shfl_xor_sync(0xffffffffu, c, s);
        if (lane == 0 && c) atomicAdd((unsigned long long *)&st->remaining, (unsigned long long)c);
    }
    grid.sync();

    uint64_t *cur = R0, *nxt = R1;
    int32_t level = (source >= 0) ? 2 : 1;
    long long left = *(volatile long long *)&st->remaining;
    while (left > 0) {
        for (int64_t w = tid; w < stride; w += nthreads) nxt[w] = cur[w];
        grid.sync();
        long long found = 0;
        for (int64_t k = warp; k < N; k += nwarps) {
            if (!((cur[k >> 6] >> (k & 63)) & 1)) continue;
            // does any predecessor of k remain?  words k>>6 down to 0, 32 at a time
            const uint64_t *row = bitsT + k * stride;
            bool blocked = false;
            for (int64_t hi = k >> 6; hi >= 0 && !blocked; hi -= 32) {
                const int64_t w = hi - lane;
                const uint64_t x = (w >= 0) ? (row[w] & cur[w]) : 0ULL;
                blocked = __any_sync(0xffffffffu, x != 0);
            }
            if (!blocked) {
                if (lane == 0) {
                    height[k] = level;
                    atomicAnd((unsigned long long *)&nxt[k >> 6], ~(1ULL << (k & 63)));
                }
                found++;
            }
        }
        if (lane == 0 && found) {
            atomicAdd((unsigned long long *)&st->remaining, (unsigned long long)(-found));
            atomicMax(&st->longest, (long long)level);
        }
        grid.sync();
        uint64_t *t = cur; cur = nxt; nxt = t;
        level++;
        const long long now = *(volatile long long *)&st->remaining;
        if (now == left) break;      // no progress: bits/bitsT are not an acyclic relation and its transpose
        left = now;
    }
    if (tid == 0 && longest_out) *longest_out = st->longest;
}

__global__ void __launch_bounds__(POSET_THREADS)
k_greedy_antichain(const uint64_t *__restrict__ bits, const uint64_t *__restrict__ bitsT, int64_t N, int64_t stride,
                   int64_t seed, uint64_t *A, uint64_t *Xi, PosetState *st, long long *size_out)
{
    cg::grid_group grid = cg::this_grid();
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nthreads = (int64_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    const int64_t warp = tid >> 5, nwarps = nthreads >> 5;
    const int64_t words = (N + 63) >> 6;

    // Xi = P \ J(seed) \ {seed},  A = {seed} | Xi
    for (int64_t w = tid; w < stride; w += nthreads) {
        const uint64_t all = w < words ? ((w == words - 1 && (N & 63)) ? (~0ULL >> (64 - (N & 63))) : ~0ULL) : 0ULL;
        const uint64_t self = (w == (seed >> 6)) ? (1ULL << (seed & 63)) : 0ULL;
        const uint64_t x = all & ~(bits[seed * stride + w] | bitsT[seed * stride + w] | self);
        Xi[w] = x;
        A[w] = x | self;
    }
    if (tid == 0) st->best[0] = st->best[1] = 0;
    grid.sync();

    for (int it = 0;; it++) {
        unsigned long long *best = &st->best[it & 1];
        // c(j) = |A \ J(j)| for every candidate; first j with the largest c
        for (int64_t j = warp; j < N; j += nwarps) {
            if (!((Xi[j >> 6] >> (j & 63)) & 1)) continue;
            const uint64_t *ru = bits + j * stride, *rl = bitsT + j * stride;
            unsigned int c = 0;
            for (int64_t w = lane; w < words; w += 32) c += __popcll(A[w] & ~(ru[w] | rl[w]));
            for (int s = 16; s >= 1; s >>= 1) c += __shfl_xor_sync(0xffffffffu, c, s);
            if (lane == 0) atomicMax(best, ((unsigned long long)c << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)j));
        }
        grid.sync();
        const unsigned long long b = *(volatile unsigned long long *)best;
        if (b == 0) break;                                   // no candidate left
        const int64_t k = (int64_t)(0xFFFFFFFFu - (unsigned int)(b & 0xFFFFFFFFu));
        for (int64_t w = tid; w < stride; w += nthreads) {
            const uint64_t Jk = bits[k * stride + w] | bitsT[k * stride + w];
            const uint64_t self = (w == (k >> 6)) ? (1ULL << (k & 63)) : 0ULL;
            A[w] &= ~Jk;
            Xi[w] &= ~(Jk | self);
        }
        if (tid == 0) st->best[(it + 1) & 1] = 0;            // last read two barriers ago
        grid.sync();
    }
    // |A|
    if (tid == 0) st->longest = 0;
    grid.sync();
    long long c = 0;
    for (int64_t w = tid; w < stride; w += nthreads) c += __popcll(A[w]);
    for (int s = 16; s >= 1; s >>= 1) c += __shfl_xor_sync(0xffffffffu, c, s);
    if (lane == 0 && c) atomicAdd((unsigned long long *)&st->longest, (unsigned long long)c);
    grid.sync();
    if (tid == 0 && size_out) *size_out = st->longest;
}

template <typename K>
int coop_grid(K kernel, int *blocks)
{
    int dev = 0, coop = 0, per_sm = 0;
    CS_CUDA(cudaGetDevice(&dev));
    CS_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    if (!coop) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "device does not support cooperative launches");
        return CS_ERR_CUDA;
    }
    CS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, POSET_THREADS, 0));
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 4) per_sm = 4;
    *blocks = sm_count() * per_sm;
    return CS_OK;
}

}  // namespace

size_t poset_workspace_bytes(int64_t N)
{
    return 256 + 2 * align_up((size_t)row_stride_words(N) * 8, 256);
}

int launch_chain_heights(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t source,
                         int32_t *height, int64_t *longest, void *ws, cudaStream_t st)
{
    int64_t stride = row_stride_words(N);
    unsigned char *p = static_cast<unsigned char *>(ws);
    PosetState *state = reinterpret_cast<PosetState *>(p);
    uint64_t *R0 = reinterpret_cast<uint64_t *>(p + 256);
    uint64_t *R1 = reinterpret_cast<uint64_t *>(p + 256 + align_up((size_t)stride * 8, 256));
    int blocks = 0;
    int rc = coop_grid(k_chain_heights, &blocks);
    if (rc) return rc;
    long long *lo = reinterpret_cast<long long *>(longest);
    void *args[] = {&bits, &bitsT, &N, &stride, &source, &height, &R0, &R1, &state, &lo};
    CS_CUDA(cudaLaunchCooperativeKernel((const void *)k_chain_heights, dim3(blocks), dim3(POSET_THREADS), args, 0, st));
    CS_LAUNCHED("k_chain_heights");
    return CS_OK;
}

int launch_greedy_antichain(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t seed,
                            uint64_t *member, int64_t *size, void *ws, cudaStream_t st)
{
    int64_t stride = row_stride_words(N);
    unsigned char *p = static_cast<unsigned char *>(ws);
    PosetState *state = reinterpret_cast<PosetState *>(p);
    uint64_t *Xi = reinterpret_cast<uint64_t *>(p + 256);
    int blocks = 0;
    int rc = coop_grid(k_greedy_antichain, &blocks);
    if (rc) return rc;
    long long *so = reinterpret_cast<long long *>(size);
    void *args[] = {&bits, &bitsT, &N, &stride, &seed, &member, &Xi, &state, &so};
    CS_CUDA(cudaLaunchCooperativeKernel((const void *)k_greedy_antichain, dim3(blocks), dim3(POSET_THREADS), args, 0, st));
    CS_LAUNCHED("k_greedy_antichain");
    return CS_OK;
}

}  // namespace cs
