// cs_common.cuh -- shared declarations of the CUDA side of libcausalset.so (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <stdio.h>
#include <string.h>

#include "../../include/causalset.h"

namespace cs {

extern thread_local char g_cuda_err[256];
extern std::atomic<long long> g_launches;   // kernels launched by this library (host counter)

inline int cuda_fail(cudaError_t e, const char *what)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
    return CS_ERR_CUDA;
}

#define CS_CUDA(call)                                               \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return cs::cuda_fail(e__, #call);   \
    } while (0)

#define CS_LAUNCHED(name)                                           \
    do {                                                            \
        cs::g_launches++;                                           \
        cudaError_t e__ = cudaGetLastError();                       \
        if (e__ != cudaSuccess) return cs::cuda_fail(e__, name);    \
    } while (0)

inline int64_t row_stride_words(int64_t N)
{
    int64_t w = (N + 63) / 64;
    return w + (w & 1);
}

inline int64_t clamp_kmax(int64_t N, int64_t kmax)
{
    int64_t top = N - 2;
    if (top < 0) top = 0;
    if (kmax < 0 || kmax > top) kmax = top;
    return kmax;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Per-device host state.  The library may be called from several threads and on several devices of one
// process: everything cached on the host is keyed by the current device, and one-time set-up that is
// idempotent (cudaFuncSetAttribute) is guarded by an atomic flag per device rather than a lock.
constexpr int MAX_DEVICES = 64;
inline int current_device()
{
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= MAX_DEVICES) d = 0;
    return d;
}
struct PerDeviceFlag {
    std::atomic<bool> done[MAX_DEVICES];
    bool get(int dev) const { return done[dev].load(std::memory_order_acquire); }
    void set(int dev) { done[dev].store(true, std::memory_order_release); }
};

int sm_count();   // SMs of the current device (cached per device)

// true while `st` is being captured into a CUDA graph (or the query itself fails, which a capture elsewhere can cause):
// the one-time self-checks synchronise the stream and take pool memory, which would invalidate the caller's capture,
// so they do not run then and the AUTO routes take the path that needs no trust for that call
inline bool stream_is_capturing(cudaStream_t st)
{
    cudaStreamCaptureStatus status = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &status) != cudaSuccess) {
        cudaGetLastError();
        return true;
    }
    return status != cudaStreamCaptureStatusNone;
}

// First 256 bytes of every a2 workspace: scheduling counters of the route and what the launch executed
// (read back through cs_interval_hist_stats).
struct IntervalStats {
    unsigned long long sched[4];          // route-private (POPC: the tile counter)
    unsigned long long stages_executed;   // (tile, 256-k stage) pairs whose MMAs were issued (pair route)
    unsigned long long stages_total;      // the same count with no empty block skipped
    unsigned long long blocks_empty;      // empty 256 x 256 bit blocks among those examined (pair route)
    unsigned long long blocks_examined;
};
static_assert(sizeof(IntervalStats) <= 256, "stats block");

// ---- stage launchers (defined in the .cu files) ---------------------------------------------
// a1.  route: CS_A1_AUTO / CS_A1_FMA / CS_A1_TENSOR; scratch (device, causal_matrix_scratch_bytes) may be NULL: the
// tensor route then takes it from the library's stream-ordered pool.
int launch_causal_matrix(const double *coords, int64_t B, int64_t N, int dim, int geometry, int route,
                         uint64_t *bits, uint64_t *bitsT, void *scratch, size_t scratch_bytes, cudaStream_t st);
size_t causal_matrix_scratch_bytes(int64_t B, int64_t N, int dim, int geometry, int route);
int tensor_route_trusted(cudaStream_t st, bool *trusted);   // one-time self-check of the tensor a1 route on this device
int interval_pair_trusted(cudaStream_t st, bool *trusted);  // the same for the tensor a2 route (cs_selfcheck.cu)
int scratch_pool(cudaMemPool_t *out);                       // the library's stream-ordered pool on the current device (cs_build.cu)
bool causal_tc_supported(int geometry, int dim);
size_t causal_tc_scratch_bytes(int64_t B, int64_t N, int dim, int geometry);
int launch_causal_tc(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                     uint64_t *bits, uint64_t *bitsT, void *scratch, cudaStream_t st);
int launch_causal_tc_probe(const double *coords, int64_t N, int dim, uint64_t *bits, uint64_t *bitsT,
                           void *scratch, double *out_host, cudaStream_t st);
int launch_transpose_bits(const uint64_t *bits, int64_t B, int64_t N, uint64_t *bitsT, cudaStream_t st);
int launch_degrees(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t *outdeg, int64_t *indeg, cudaStream_t st);
int launch_relation_stats(const uint64_t *bits, int64_t N, int64_t *out, cudaStream_t st);

// hist (int64[B][kmax+1]) and nrel (int64[B] or NULL) must be zeroed by the caller.
int launch_interval_popc(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                         int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                         void *scratch, cudaStream_t st);
size_t interval_popc_scratch_bytes();
// the bit route with its scratch in a static device array (no allocation anywhere on the path); N <= interval_static_max_n()
int launch_interval_popc_static(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                                int64_t *hist, int64_t *nrel, cudaStream_t st);
int64_t interval_static_max_n();

int launch_interval_tensor(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                           int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                           void *scratch, size_t scratch_bytes, cudaStream_t st);
size_t interval_tensor_scratch_bytes(int64_t B, int64_t N);
int launch_interval_fp4(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                        int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                        void *scratch, size_t scratch_bytes, cudaStream_t st);
// keep_table: the tile table in `scratch` was written by an earlier call with the same N on this stream (the chunks of an
// ensemble): it is not rebuilt.
int launch_interval_pair(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                         int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                         void *scratch, size_t scratch_bytes, IntervalStats *stats, bool keep_table, cudaStream_t st);
size_t interval_pair_scratch_bytes(int64_t N);
bool interval_tensor_available();

int launch_bd_action(const int64_t *hist, int64_t hist_stride, int64_t B, int64_t kmax, int64_t N, int dim,
                     double *action, int64_t *bracket, int64_t *hist4, cudaStream_t st);

int launch_peak_probe(int kind, int64_t iters, void *workspace, size_t workspace_bytes, double *out_host, cudaStream_t st);

size_t poset_workspace_bytes(int64_t N);
int launch_chain_heights(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t source,
                         int32_t *height, int64_t *longest, void *ws, cudaStream_t st);
int launch_greedy_antichain(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t seed,
                            uint64_t *member, int64_t *size, void *ws, cudaStream_t st);
int launch_smeared_action(const int64_t *hist, int64_t hist_stride, int64_t B, int64_t kmax, int64_t N, int dim,
                          double eps, double *action, cudaStream_t st);

}  // namespace cs
