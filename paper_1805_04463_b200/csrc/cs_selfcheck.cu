// cs_selfcheck.cu -- one-time self-check of the tensor-core a2 route on a device (behind CS_ROUTE_AUTO).
//
// k_interval_pair (cs_interval_pair.cu) reads its counts straight from the bit pattern of fp32 accumulators that hold
// SUBNORMAL numbers: block scales of 2^-72 .. 2^-74 make every product 2^-146 = 8 units of 2^-149, and the pattern of
// the sum is the integer 8 * count.  That is exact only if tcgen05.mma neither flushes subnormal products or partial
// sums to zero nor rounds them -- measured behaviour of the B200 this was written on, stated nowhere (DESIGN.md,
// reading A22).  A part, driver or firmware that flushes would hand back wrong histograms without any error, so the
// first time CS_ROUTE_AUTO would pick that route on a device the library checks it there:
//   1. a total order of 2048 + 77 elements (several tiles, a ragged tail): the histogram has the closed form
//      N_k = N - 1 - k (PAPER.md:1755-1758 with every pair related), and the pair (i, j) has count j - i - 1, so every
//      count 0 .. N-2 occurs -- a flushed sum, a lost K stage or a wrong scale cannot hide;
//   2. a seeded 3+1 flat-cone causet of the same size against the AND/POPC route, whole histogram, and once more with
//      kmax = 3 (the ensemble variant of the kernel, which shifts the pattern instead of converting it).
// On any mismatch AUTO keeps the POPC route on that device (CS_ROUTE_TENSOR_PAIR still runs when asked for by name) and
// cs_last_cuda_error() says what differed.  Costs ~1 ms, a pool allocation of ~2 MiB and one stream synchronisation, once.
#include <mutex>
#include <vector>

#include "cs_common.cuh"

namespace cs {

namespace {

// chain: (t, x) = (i, 0), every pair related under the flat cone; else SplitMix64 points of a 3+1 box, time increasing
__global__ void k_a2check_coords(double *coords, int N, int dim, int chain)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (chain) {
        coords[(size_t)i * dim] = (double)i;
        for (int d = 1; d < dim; d++) coords[(size_t)i * dim + d] = 0.0;
        return;
    }
    coords[(size_t)i * dim] = -0.9 + 1.8 * (i + 0.5) / N;
    uint64_t z = 0xD1B54A32D192ED03ull * (uint64_t)(i + 1);
    for (int d = 1; d < dim; d++) {
        z += 0x9E3779B97F4A7C15ull;
        uint64_t x = z;
        x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
        x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
        x ^= x >> 31;
        coords[(size_t)i * dim + d] = ((double)(x >> 11) * 0x1p-53 - 0.5) * 0.9;
    }
}

struct CheckBuffers {
    double *coords;
    uint64_t *bits, *bitsT;
    int64_t *hist_pair, *hist_popc;
    IntervalStats *stats;
    void *pair_scratch;
    size_t pair_scratch_bytes;
};

int run_case(const CheckBuffers &b, int64_t N, int dim, bool chain, int64_t kmax, std::vector<int64_t> &h_pair,
             std::vector<int64_t> &h_popc, cudaStream_t st)
{
    const size_t hb = (size_t)(kmax + 1) * sizeof(int64_t);
    k_a2check_coords<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(b.coords, (int)N, dim, chain ? 1 : 0);
    CS_LAUNCHED("k_a2check_coords");
    int rc = launch_causal_matrix(b.coords, 1, N, dim, CS_GEOM_MINK_CONE, CS_A1_FMA, b.bits, b.bitsT, nullptr, 0, st);
    if (rc) return rc;
    CS_CUDA(cudaMemsetAsync(b.hist_pair, 0, hb, st));
    CS_CUDA(cudaMemsetAsync(b.hist_popc, 0, hb, st));
    CS_CUDA(cudaMemsetAsync(b.stats, 0, 256, st));
    rc = launch_interval_pair(b.bits, b.bitsT, 1, N, kmax, 0, N, b.hist_pair, nullptr, b.pair_scratch, b.pair_scratch_bytes,
                              b.stats, false, st);
    if (rc) return rc;
    CS_CUDA(cudaMemsetAsync(b.stats, 0, 256, st));
    rc = launch_interval_popc(b.bits, b.bitsT, 1, N, kmax, 0, N, b.hist_popc, nullptr, b.stats, st);
    if (rc) return rc;
    h_pair.assign((size_t)kmax + 1, -1);
    h_popc.assign((size_t)kmax + 1, -2);
    CS_CUDA(cudaMemcpyAsync(h_pair.data(), b.hist_pair, hb, cudaMemcpyDeviceToHost, st));
    CS_CUDA(cudaMemcpyAsync(h_popc.data(), b.hist_popc, hb, cudaMemcpyDeviceToHost, st));
    CS_CUDA(cudaStreamSynchronize(st));
    return CS_OK;
}

}  // namespace

int interval_pair_trusted(cudaStream_t st, bool *trusted)
{
    static std::atomic<int> state[MAX_DEVICES];       // 0 not checked, 1 counts are exact, 2 they are not
    static std::mutex mu;
    const int dev = current_device();
    int s0 = state[dev].load(std::memory_order_acquire);
    if (s0 == 0 && stream_is_capturing(st)) {         // not now: the check would break the caller's capture
        *trusted = false;
        return CS_OK;
    }
    if (s0 == 0) {
        std::lock_guard<std::mutex> lock(mu);
        s0 = state[dev].load(std::memory_order_acquire);
        if (s0 == 0) {
            cudaMemPool_t pool;
            int rc = scratch_pool(&pool);
            if (rc) return rc;
            const int64_t N = 2048 + 77, stride = row_stride_words(N), kfull = N - 2;
            const size_t cb = align_up((size_t)N * 4 * 8, 256), mb = align_up((size_t)N * stride * 8, 256);
            const size_t hb = align_up((size_t)(kfull + 1) * 8, 256), ps = align_up(interval_pair_scratch_bytes(N), 256);
            unsigned char *p = nullptr;
            CS_CUDA(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&p), cb + 2 * mb + 2 * hb + 256 + ps, pool, st));
            CheckBuffers b;
            b.coords = reinterpret_cast<double *>(p);
            b.bits = reinterpret_cast<uint64_t *>(p + cb);
            b.bitsT = reinterpret_cast<uint64_t *>(p + cb + mb);
            b.hist_pair = reinterpret_cast<int64_t *>(p + cb + 2 * mb);
            b.hist_popc = reinterpret_cast<int64_t *>(p + cb + 2 * mb + hb);
            b.stats = reinterpret_cast<IntervalStats *>(p + cb + 2 * mb + 2 * hb);
            b.pair_scratch = p + cb + 2 * mb + 2 * hb + 256;
            b.pair_scratch_bytes = ps;
            bool ok = true;
            char why[200] = "";
            rc = [&]() -> int {                           // every exit passes the cudaFreeAsync below
                std::vector<int64_t> hp, hq;
                int r = run_case(b, N, 2, true, kfull, hp, hq, st);
                if (r) return r;
                for (int64_t k = 0; k <= kfull && ok; k++)
                    if (hp[k] != N - 1 - k || hq[k] != N - 1 - k) {
                        ok = false;
                        snprintf(why, sizeof(why), "total order of %lld: N_%lld = %lld (tensor route), %lld (POPC route), closed form %lld",
                                 (long long)N, (long long)k, (long long)hp[k], (long long)hq[k], (long long)(N - 1 - k));
                    }
                if (!ok) return CS_OK;
                for (int pass = 0; pass < 2 && ok; pass++) {
                    const int64_t kmax = pass == 0 ? kfull : 3;
                    r = run_case(b, N, 4, false, kmax, hp, hq, st);
                    if (r) return r;
                    int64_t total = 0;
                    for (int64_t k = 0; k <= kmax && ok; k++) {
                        total += hp[k];
                        if (hp[k] != hq[k]) {
                            ok = false;
                            snprintf(why, sizeof(why), "3+1 causet of %lld, kmax %lld: N_%lld = %lld (tensor route), %lld (POPC route)",
                                     (long long)N, (long long)kmax, (long long)k, (long long)hp[k], (long long)hq[k]);
                        }
                    }
                    if (ok && total == 0) {
                        ok = false;
                        snprintf(why, sizeof(why), "3+1 causet of %lld: empty histogram", (long long)N);
                    }
                }
                return CS_OK;
            }();
            cudaFreeAsync(p, st);
            if (rc) return rc;
            if (!ok)
                snprintf(g_cuda_err, sizeof(g_cuda_err), "a2 self-check failed on device %d (%s): CS_ROUTE_AUTO keeps the POPC route", dev, why);
            s0 = ok ? 1 : 2;
            state[dev].store(s0, std::memory_order_release);
        }
    }
    *trusted = s0 == 1;
    return CS_OK;
}

}  // namespace cs
