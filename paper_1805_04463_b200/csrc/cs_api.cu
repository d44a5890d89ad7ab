// cs_api.cu -- the extern "C" boundary of libcausalset.so (include/causalset.h).
// Argument checking, workspace carving and kernel sequencing only; the arithmetic lives in
// cs_poset.cu (NEXT-3), cs_build.cu (a1), cs_selfcheck.cu (the a2 self-check), cs_interval_popc.cu / cs_interval_tensor.cu / cs_interval_fp4.cu / cs_interval_pair.cu (a2) and cs_action.cu (a3).
#include <mutex>

#include "cs_common.cuh"

namespace cs {

thread_local char g_cuda_err[256] = "";
std::atomic<long long> g_launches{0};

int sm_count()
{
    static std::atomic<int> cached[MAX_DEVICES];
    const int dev = current_device();
    int n = cached[dev].load(std::memory_order_relaxed);
    if (n <= 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
        cached[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

// spacetime dimension of a point set: the number of coordinates, except for the FLRW geometry whose six
// numbers per point describe a 3+1 dimensional event
static int spacetime_dim(int geometry, int dim)
{
    return (geometry == CS_GEOM_FLRW_POLAR || geometry == CS_GEOM_DS4_SPHERICAL) ? 4 : dim;
}

// rows are read with 128-bit loads, bulk copies and TMA: the matrices must start on a 16-byte boundary
static bool misaligned16(const void *a, const void *b)
{
    return (((uintptr_t)a | (uintptr_t)b) & 15) != 0;
}

static int resolve_route(int64_t N, int route)
{
    if (route == CS_ROUTE_AUTO) route = cs_default_route(N);
    if (route >= CS_ROUTE_TENSOR && !interval_tensor_available()) return -1;
    return route;
}

static size_t interval_ws_bytes(int64_t B, int64_t N, int have_bitsT, int route)
{
    size_t ws = 256;   // tile counter etc.
    if (!have_bitsT) ws += align_up((size_t)B * N * row_stride_words(N) * 8, 256);
    if (route == CS_ROUTE_TENSOR) ws += align_up(interval_tensor_scratch_bytes(B, N), 256);
    if (route == CS_ROUTE_TENSOR_PAIR) ws += align_up(interval_pair_scratch_bytes(N), 256);
    return ws;
}

// hist: int64[B][kmax+1]; shared by the single and the batched entry points
static int interval_hist_impl(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                              int64_t row_begin, int64_t row_end, int route, int64_t *hist, int64_t *nrel,
                              void *workspace, size_t workspace_bytes, cudaStream_t st, bool keep_table = false)
{
    kmax = clamp_kmax(N, kmax);
    CS_CUDA(cudaMemsetAsync(hist, 0, (size_t)B * (kmax + 1) * sizeof(int64_t), st));
    if (nrel) CS_CUDA(cudaMemsetAsync(nrel, 0, sizeof(int64_t), st));
    if (N < 2) return CS_OK;
    if (row_begin < 0) row_begin = 0;
    if (row_end > N) row_end = N;
    if (row_begin >= row_end) return CS_OK;
    const bool by_default = route == CS_ROUTE_AUTO;
    route = resolve_route(N, route);
    if (route < 0) return CS_ERR_ARG;
    if (by_default && route == CS_ROUTE_TENSOR_PAIR) {
        // the tensor route reads integers out of subnormal accumulators (reading A22): checked once per
        // device; a device that fails the check -- or on which it could not run -- gets the bit route
        bool trusted = false;
        if (interval_pair_trusted(st, &trusted) != CS_OK) {
            cudaGetLastError();
            trusted = false;
        }
        if (!trusted) route = CS_ROUTE_POPC;
    }
    const size_t need = interval_ws_bytes(B, N, bitsT != nullptr, route);
    if (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 255)) return CS_ERR_WORKSPACE;
    unsigned char *ws = static_cast<unsigned char *>(workspace);
    void *scratch = ws;
    CS_CUDA(cudaMemsetAsync(scratch, 0, 256, st));   // IntervalStats
    ws += 256;
    if (!bitsT) {
        uint64_t *t = reinterpret_cast<uint64_t *>(ws);
        ws += align_up((size_t)B * N * row_stride_words(N) * 8, 256);
        int rc = launch_transpose_bits(bits, B, N, t, st);
        if (rc) return rc;
        bitsT = t;
    }
    if (route == CS_ROUTE_TENSOR_PAIR)
        return launch_interval_pair(bits, bitsT, B, N, kmax, row_begin, row_end, hist, nrel, ws,
                                    workspace_bytes - (size_t)(ws - static_cast<unsigned char *>(workspace)),
                                    static_cast<IntervalStats *>(scratch), keep_table, st);
    if (route == CS_ROUTE_TENSOR_FP4)
        return launch_interval_fp4(bits, bitsT, B, N, kmax, row_begin, row_end, hist, nrel, ws,
                                   workspace_bytes - (size_t)(ws - static_cast<unsigned char *>(workspace)), st);
    if (route == CS_ROUTE_TENSOR)
        return launch_interval_tensor(bits, bitsT, B, N, kmax, row_begin, row_end, hist, nrel, ws,
                                      workspace_bytes - (size_t)(ws - static_cast<unsigned char *>(workspace)), st);
    return launch_interval_popc(bits, bitsT, B, N, kmax, row_begin, row_end, hist, nrel, scratch, st);
}

}  // namespace cs

using namespace cs;

extern "C" {

const char *cs_version(void) { return "causalset-b200 0.1 (sm_100a)"; }

const char *cs_status_string(int status)
{
    switch (status) {
    case CS_OK: return "ok";
    case CS_ERR_ARG: return "invalid argument";
    case CS_ERR_DIM: return "dimension not valid for this geometry/action";
    case CS_ERR_GEOM: return "unknown geometry";
    case CS_ERR_UNSORTED: return "elements not sorted by time";
    case CS_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case CS_ERR_CUDA: return "CUDA error";
    case CS_ERR_CAPACITY: return "size beyond the fixed capacity of this entry point";
    default: return "unknown status";
    }
}

const char *cs_last_cuda_error(void) { return g_cuda_err; }

int64_t cs_row_stride_words(int64_t N) { return N < 0 ? 0 : row_stride_words(N); }

int64_t cs_launch_count(void) { return g_launches.load(); }

int cs_peak_probe(int kind, int64_t iters, void *workspace, size_t workspace_bytes, double *out_host, void *stream)
{
    if (!out_host) return CS_ERR_ARG;
    return launch_peak_probe(kind, iters, workspace, workspace_bytes, out_host, static_cast<cudaStream_t>(stream));
}

int cs_default_route(int64_t N)
{
    // measured on B200: the 4-bit tensor route on CTA pairs wins from N ~ 1024 up (12.5 ms
    // against 20.3 ms single-CTA and 327 ms POPC at N = 65536); below that a few 256 x 256 tiles cannot
    // fill the machine and the bit route is as fast
    // beyond N = 2^21 the tensor route's 8 * count no longer fits the exact range of its accumulators: bit route
    return interval_tensor_available() && N >= 1024 && N <= ((int64_t)1 << 21) ? CS_ROUTE_TENSOR_PAIR : CS_ROUTE_POPC;
}

static int check_a1_args(const double *coords, int64_t B, int64_t N, int dim, int geometry, const uint64_t *bits)
{
    if (N < 0 || B < 0) return CS_ERR_ARG;
    if (geometry < CS_GEOM_MINK2_LIGHTCONE || geometry > CS_GEOM_DS4_SPHERICAL) return CS_ERR_GEOM;
    const int want = geometry == CS_GEOM_FLRW_POLAR ? 6 : geometry == CS_GEOM_DS4_SPHERICAL ? 7 : 2;
    if (geometry == CS_GEOM_MINK_CONE ? (dim < 2 || dim > 5) : (dim != want)) return CS_ERR_DIM;
    if (N == 0 || B == 0) return 1;      // nothing to do
    if (!coords || !bits) return CS_ERR_ARG;
    return CS_OK;
}

// a1 -> a2 -> a3 entry points: the arguments of a1 and a spacetime dimension the action is defined for (Eq. 4.10-4.12:
// 2, 3, 4), checked before any work is enqueued
static int check_pipeline_args(int64_t N, int dim, int geometry)
{
    const int rc = check_a1_args(reinterpret_cast<const double *>(16), 1, N > 0 ? N : 1, dim, geometry,
                                 reinterpret_cast<const uint64_t *>(16));
    if (rc < 0) return rc;
    const int sd = spacetime_dim(geometry, dim);
    return (sd < 2 || sd > 4) ? CS_ERR_DIM : CS_OK;
}

size_t cs_causal_matrix_workspace(int64_t B, int64_t N, int dim, int geometry, int route)
{
    if (check_a1_args(reinterpret_cast<const double *>(16), B, N, dim, geometry, reinterpret_cast<const uint64_t *>(16)) != CS_OK) return 0;
    if (route < CS_A1_AUTO || route > CS_A1_TENSOR) return 0;
    return causal_matrix_scratch_bytes(B, N, dim, geometry, route);
}

int cs_default_a1_route(int64_t B, int64_t N, int dim, int geometry)
{
    if (B < 1 || N < 1) return CS_A1_FMA;
    return causal_matrix_scratch_bytes(B, N, dim, geometry, CS_A1_AUTO) ? CS_A1_TENSOR : CS_A1_FMA;
}

int cs_causal_matrix_ex(const double *coords, int64_t B, int64_t N, int dim, int geometry, int route,
                        uint64_t *bits, uint64_t *bitsT, void *workspace, size_t workspace_bytes, void *stream)
{
    const int rc = check_a1_args(coords, B, N, dim, geometry, bits);
    if (rc) return rc < 0 ? rc : CS_OK;
    if (route < CS_A1_AUTO || route > CS_A1_TENSOR) return CS_ERR_ARG;
    if (misaligned16(bits, bitsT)) return CS_ERR_ARG;
    return launch_causal_matrix(coords, B, N, dim, geometry, route, bits, bitsT, workspace, workspace_bytes,
                                static_cast<cudaStream_t>(stream));
}

int cs_causal_matrix_batched(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                             uint64_t *bits, uint64_t *bitsT, void *stream)
{
    return cs_causal_matrix_ex(coords, B, N, dim, geometry, CS_A1_AUTO, bits, bitsT, nullptr, 0, stream);
}

int cs_causal_matrix(const double *coords, int64_t N, int dim, int geometry,
                     uint64_t *bits, uint64_t *bitsT, void *stream)
{
    return cs_causal_matrix_ex(coords, 1, N, dim, geometry, CS_A1_AUTO, bits, bitsT, nullptr, 0, stream);
}

int cs_a1_tensor_selfcheck(void *stream)
{
    bool trusted = false;
    const int rc = tensor_route_trusted(static_cast<cudaStream_t>(stream), &trusted);
    return rc ? rc : (trusted ? 1 : 0);
}

int cs_a2_tensor_selfcheck(void *stream)
{
    bool trusted = false;
    const int rc = interval_pair_trusted(static_cast<cudaStream_t>(stream), &trusted);
    return rc ? rc : (trusted ? 1 : 0);
}

int cs_a1_tensor_probe(const double *coords, int64_t N, int dim, uint64_t *bits, uint64_t *bitsT,
                       void *workspace, size_t workspace_bytes, double *out_host, void *stream)
{
    if (!coords || !bits || !out_host || N < 256) return CS_ERR_ARG;     // the tensor route wants rows of >= 32 bytes
    if (dim != 4 && dim != 5) return CS_ERR_DIM;
    if (misaligned16(bits, bitsT)) return CS_ERR_ARG;
    if (!causal_tc_supported(CS_GEOM_MINK_CONE, dim)) return CS_ERR_ARG;
    if (!workspace || workspace_bytes < causal_tc_scratch_bytes(1, N, dim, CS_GEOM_MINK_CONE) || ((uintptr_t)workspace & 255))
        return CS_ERR_WORKSPACE;
    return launch_causal_tc_probe(coords, N, dim, bits, bitsT, workspace, out_host, static_cast<cudaStream_t>(stream));
}

int cs_transpose_bits(const uint64_t *bits, int64_t N, uint64_t *bitsT, void *stream)
{
    if (N < 0) return CS_ERR_ARG;
    if (N == 0) return CS_OK;
    if (!bits || !bitsT) return CS_ERR_ARG;
    return launch_transpose_bits(bits, 1, N, bitsT, static_cast<cudaStream_t>(stream));
}

int cs_relation_stats(const uint64_t *bits, int64_t N, int64_t *out, void *stream)
{
    if (N < 0 || !out || (N > 0 && !bits)) return CS_ERR_ARG;
    return launch_relation_stats(bits, N, out, static_cast<cudaStream_t>(stream));
}

int cs_degrees(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t *outdeg, int64_t *indeg, void *stream)
{
    if (N < 0 || (N > 0 && !bits) || (indeg && N > 0 && !bitsT)) return CS_ERR_ARG;
    return launch_degrees(bits, indeg ? bitsT : nullptr, N, outdeg, indeg, static_cast<cudaStream_t>(stream));
}

size_t cs_interval_hist_workspace(int64_t N, int64_t kmax, int have_bitsT, int route)
{
    (void)kmax;
    if (N < 0) return 0;
    int r = resolve_route(N, route);
    if (r < 0) r = CS_ROUTE_POPC;
    return interval_ws_bytes(1, N, have_bitsT, r);
}

int cs_interval_hist_ex(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                        int64_t row_begin, int64_t row_end, int route,
                        int64_t *hist, int64_t *n_relations,
                        void *workspace, size_t workspace_bytes, void *stream)
{
    if (N < 0 || !hist || (N > 0 && !bits)) return CS_ERR_ARG;
    if (route < CS_ROUTE_AUTO || route > CS_ROUTE_TENSOR_PAIR) return CS_ERR_ARG;
    if (misaligned16(bits, bitsT)) return CS_ERR_ARG;
    return interval_hist_impl(bits, bitsT, 1, N, kmax, row_begin, row_end, route, hist, n_relations,
                              workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
}

size_t cs_interval_hist_batched_workspace(int64_t B, int64_t N, int route)
{
    if (N < 0 || B < 0) return 0;
    int r = resolve_route(N, route);
    if (r < 0) r = CS_ROUTE_POPC;
    return interval_ws_bytes(B, N, 1, r);
}

int cs_interval_hist_batched(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                             int route, int64_t *hist, void *workspace, size_t workspace_bytes, void *stream)
{
    if (N < 0 || B < 0 || !hist) return CS_ERR_ARG;
    if (B == 0) return CS_OK;
    if (N > 0 && (!bits || !bitsT)) return CS_ERR_ARG;
    if (route < CS_ROUTE_AUTO || route > CS_ROUTE_TENSOR_PAIR) return CS_ERR_ARG;
    if (misaligned16(bits, bitsT)) return CS_ERR_ARG;
    return interval_hist_impl(bits, bitsT, B, N, kmax, 0, N, route, hist, nullptr,
                              workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
}

int cs_interval_hist(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                     int64_t *hist, int64_t *n_relations,
                     void *workspace, size_t workspace_bytes, void *stream)
{
    return cs_interval_hist_ex(bits, bitsT, N, kmax, 0, N, CS_ROUTE_AUTO, hist, n_relations,
                               workspace, workspace_bytes, stream);
}

int64_t cs_interval_hist_static_max_n(void) { return interval_static_max_n(); }

int cs_interval_hist_static(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                            int64_t *hist, int64_t *n_relations, void *stream)
{
    if (N < 0 || !hist || (N > 0 && !bits)) return CS_ERR_ARG;
    if (misaligned16(bits, bitsT)) return CS_ERR_ARG;
    return launch_interval_popc_static(bits, bitsT, N, kmax, hist, n_relations, static_cast<cudaStream_t>(stream));
}

int cs_interval_hist_stats(const void *workspace, int64_t *stats_host, void *stream)
{
    if (!workspace || !stats_host || ((uintptr_t)workspace & 255)) return CS_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    IntervalStats h;
    CS_CUDA(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, st));
    CS_CUDA(cudaStreamSynchronize(st));
    stats_host[0] = (int64_t)h.stages_executed;
    stats_host[1] = (int64_t)h.stages_total;
    stats_host[2] = (int64_t)h.blocks_empty;
    stats_host[3] = (int64_t)h.blocks_examined;
    return CS_OK;
}

int cs_bd_action(const int64_t *hist, int64_t kmax, int64_t N, int dim,
                 double *action, int64_t *bracket, void *stream)
{
    if (!hist || !action || N < 0) return CS_ERR_ARG;
    if (dim < 2 || dim > 4) return CS_ERR_DIM;
    if (kmax < 0) kmax = clamp_kmax(N, kmax);
    return launch_bd_action(hist, kmax + 1, 1, kmax, N, dim, action, bracket, nullptr,
                            static_cast<cudaStream_t>(stream));
}

int cs_smeared_action(const int64_t *hist, int64_t kmax, int64_t N, int dim, double eps,
                      double *action, void *stream)
{
    if (!hist || !action || N < 0) return CS_ERR_ARG;
    kmax = clamp_kmax(N, kmax);
    return launch_smeared_action(hist, kmax + 1, 1, kmax, N, dim, eps, action, static_cast<cudaStream_t>(stream));
}

size_t cs_poset_workspace(int64_t N) { return N < 0 ? 0 : poset_workspace_bytes(N); }

int cs_chain_heights(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t source,
                     int32_t *height, int64_t *longest, void *workspace, size_t workspace_bytes, void *stream)
{
    if (N < 0 || source < -1 || source >= N) return CS_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (longest) CS_CUDA(cudaMemsetAsync(longest, 0, sizeof(int64_t), st));
    if (N == 0) return CS_OK;
    if (!bits || !bitsT || !height) return CS_ERR_ARG;
    if (!workspace || workspace_bytes < poset_workspace_bytes(N) || ((uintptr_t)workspace & 255)) return CS_ERR_WORKSPACE;
    return launch_chain_heights(bits, bitsT, N, source, height, longest, workspace, st);
}

int cs_greedy_antichain(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t seed,
                        uint64_t *member, int64_t *size, void *workspace, size_t workspace_bytes, void *stream)
{
    if (N <= 0 || seed < 0 || seed >= N) return CS_ERR_ARG;
    if (!bits || !bitsT || !member) return CS_ERR_ARG;
    if (!workspace || workspace_bytes < poset_workspace_bytes(N) || ((uintptr_t)workspace & 255)) return CS_ERR_WORKSPACE;
    return launch_greedy_antichain(bits, bitsT, N, seed, member, size, workspace, static_cast<cudaStream_t>(stream));
}

// ---- batched ensemble ----------------------------------------------------------------------
// The ensemble is processed in chunks of CB causets: a1 writes the chunk's bit matrices, a2 reduces them to
// N_0..N_3, and the same buffers take the next chunk, so the workspace holds the matrices of one chunk (at most
// ENSEMBLE_MAT_BYTES), not of the ensemble (4 GiB for 4096 x 2048).  CB is a whole number of causets per CTA pair
// of a2's persistent grid (causet-major schedule: every pair then gets the same number of causets).
// workspace: [bits CB*N*stride][bitsT CB*N*stride][hist B*4 int64][interval scratch]
constexpr size_t ENSEMBLE_MAT_BYTES = (size_t)500 << 20;     // both matrices of a chunk + the scratch of its a1

// a1 scratch of cb causets carved from the workspace.  The workspace queries do not know the geometry: the carve is sized
// for the K = 32 operand rows with the widest coordinates (Eq. 7.7: six doubles per point), which covers the flat cone up
// to 3+1 dimensions; the two geometries with K = 48 rows take their scratch from the library's pool instead.
static size_t ensemble_a1_scratch(int64_t cb, int64_t N)
{
    return align_up(causal_tc_scratch_bytes(cb, N, 6, CS_GEOM_FLRW_POLAR), 256);
}

static int64_t ensemble_chunk(int64_t B, int64_t N)
{
    const size_t per = 2 * (size_t)N * row_stride_words(N) * 8 + ensemble_a1_scratch(1, N);
    int64_t cb = per ? (int64_t)(ENSEMBLE_MAT_BYTES / per) : B;
    const int64_t pairs = sm_count() / 2;
    if (cb > pairs) cb -= cb % pairs;
    if (cb < 1) cb = 1;
    return cb < B ? cb : B;
}

size_t cs_bd_action_batched_workspace(int64_t B, int64_t N)
{
    if (B < 0 || N < 0) return 0;
    const int64_t CB = ensemble_chunk(B, N);
    const size_t mat = align_up((size_t)CB * N * row_stride_words(N) * 8, 256);
    int r = cs_default_route(N);
    return 2 * mat + align_up((size_t)B * 4 * 8, 256) + interval_ws_bytes(CB, N, 1, r) + ensemble_a1_scratch(CB, N);
}

int cs_bd_action_batched(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                         double *actions, int64_t *hist4,
                         void *workspace, size_t workspace_bytes, void *stream)
{
    if (B < 0 || N < 0) return CS_ERR_ARG;
    if (B == 0) return CS_OK;
    if (!coords || !actions) return CS_ERR_ARG;
    {   // geometry, dim and the action's dimension before any chunk is built
        const int rc = check_pipeline_args(N, dim, geometry);
        if (rc) return rc;
    }
    if (!workspace || workspace_bytes < cs_bd_action_batched_workspace(B, N) || ((uintptr_t)workspace & 255))
        return CS_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int64_t CB = ensemble_chunk(B, N);
    const size_t mat = align_up((size_t)CB * N * row_stride_words(N) * 8, 256);
    unsigned char *ws = static_cast<unsigned char *>(workspace);
    uint64_t *bits = reinterpret_cast<uint64_t *>(ws);
    uint64_t *bitsT = reinterpret_cast<uint64_t *>(ws + mat);
    int64_t *hist = reinterpret_cast<int64_t *>(ws + 2 * mat);
    unsigned char *iws = ws + 2 * mat + align_up((size_t)B * 4 * 8, 256);
    const size_t a1_bytes = ensemble_a1_scratch(CB, N);
    unsigned char *a1ws = ws + cs_bd_action_batched_workspace(B, N) - a1_bytes;
    const int64_t kmax = clamp_kmax(N, 3);
    // hist rows are kmax+1 long; with kmax = 3 that is the [B][4] layout asked for
    if (kmax < 3) CS_CUDA(cudaMemsetAsync(hist, 0, (size_t)B * 4 * 8, st));
    for (int64_t b0 = 0; b0 < B; b0 += CB) {
        const int64_t nb = B - b0 < CB ? B - b0 : CB;
        const bool fits = cs_causal_matrix_workspace(nb, N, dim, geometry, CS_A1_AUTO) <= a1_bytes;
        int rc = cs_causal_matrix_ex(coords + b0 * N * dim, nb, N, dim, geometry, CS_A1_AUTO, bits, bitsT, fits ? a1ws : nullptr,
                                     fits ? a1_bytes : 0, stream);
        if (rc) return rc;
        rc = interval_hist_impl(bits, bitsT, nb, N, kmax, 0, N, CS_ROUTE_AUTO, hist + b0 * (kmax + 1), nullptr, iws,
                                (size_t)(a1ws - iws), st, b0 > 0);      // the tile table of the first chunk serves them all
        if (rc) return rc;
    }
    return launch_bd_action(hist, kmax + 1, B, kmax, N, spacetime_dim(geometry, dim), actions, nullptr, hist4, st);
}

// ---- ensemble end to end with host buffers: chunked, copies overlapped with compute -------------
// The coordinates of the next chunk of causets (ensemble_chunk above) travel over PCIe on a library-owned copy
// stream while the caller's stream builds and reduces the current chunk; two coordinate buffers alternate, the
// bit matrices exist for one chunk only.
// workspace: [coords chunk x2][bits chunk][bitsT chunk][hist CB*4][actions B][hist4 B*4][interval scratch]
// copy stream and events of the host pipeline, one set per device, created under a lock on first use;
// a partial failure destroys what was created so that the next call starts over
struct CopyPipe {
    cudaStream_t stream = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr}, start = nullptr;
    bool ready = false;
};
static int copy_pipe(CopyPipe **out)
{
    static CopyPipe pipes[MAX_DEVICES];
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    CopyPipe &p = pipes[current_device()];
    if (!p.ready) {
        cudaError_t e = cudaStreamCreateWithFlags(&p.stream, cudaStreamNonBlocking);
        for (int i = 0; i < 2 && e == cudaSuccess; i++) {
            e = cudaEventCreateWithFlags(&p.copied[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p.consumed[i], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p.start, cudaEventDisableTiming);
        if (e != cudaSuccess) {
            for (int i = 0; i < 2; i++) {
                if (p.copied[i]) cudaEventDestroy(p.copied[i]);
                if (p.consumed[i]) cudaEventDestroy(p.consumed[i]);
            }
            if (p.start) cudaEventDestroy(p.start);
            if (p.stream) cudaStreamDestroy(p.stream);
            p = CopyPipe();
            return cuda_fail(e, "host pipeline set-up");
        }
        p.ready = true;
    }
    *out = &p;
    return CS_OK;
}

size_t cs_bd_action_batched_host_workspace(int64_t B, int64_t N, int dim)
{
    if (B < 0 || N < 0 || dim < 2 || dim > 7) return 0;
    const int64_t CB = ensemble_chunk(B, N);
    const size_t cbuf = align_up((size_t)CB * N * dim * 8, 256);
    const size_t mat = align_up((size_t)CB * N * row_stride_words(N) * 8, 256);
    return 2 * cbuf + 2 * mat + align_up((size_t)CB * 4 * 8, 256) + align_up((size_t)B * 8, 256) +
           align_up((size_t)B * 4 * 8, 256) + interval_ws_bytes(CB, N, 1, cs_default_route(N)) + ensemble_a1_scratch(CB, N);
}

int cs_bd_action_batched_host(const double *coords_host, int64_t B, int64_t N, int dim, int geometry,
                              double *actions_host, int64_t *hist4_host,
                              void *workspace, size_t workspace_bytes, void *stream)
{
    if (B < 0 || N < 0) return CS_ERR_ARG;
    if (B == 0) return CS_OK;
    if (!coords_host || !actions_host) return CS_ERR_ARG;
    {
        const int rc = check_pipeline_args(N, dim, geometry);
        if (rc) return rc;
    }
    if (!workspace || workspace_bytes < cs_bd_action_batched_host_workspace(B, N, dim) || ((uintptr_t)workspace & 255))
        return CS_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CopyPipe *pipe = nullptr;
    int prc = copy_pipe(&pipe);
    if (prc) return prc;
    cudaStream_t copy_stream = pipe->stream;
    cudaEvent_t *copied = pipe->copied, *consumed = pipe->consumed, start = pipe->start;
    const int64_t CB = ensemble_chunk(B, N);
    const size_t cbuf = align_up((size_t)CB * N * dim * 8, 256);
    const size_t mat = align_up((size_t)CB * N * row_stride_words(N) * 8, 256);
    unsigned char *ws = static_cast<unsigned char *>(workspace);
    double *cdev[2] = {reinterpret_cast<double *>(ws), reinterpret_cast<double *>(ws + cbuf)};
    ws += 2 * cbuf;
    uint64_t *bits = reinterpret_cast<uint64_t *>(ws);
    uint64_t *bitsT = reinterpret_cast<uint64_t *>(ws + mat);
    ws += 2 * mat;
    int64_t *hist = reinterpret_cast<int64_t *>(ws);
    ws += align_up((size_t)CB * 4 * 8, 256);
    double *actions = reinterpret_cast<double *>(ws);
    ws += align_up((size_t)B * 8, 256);
    int64_t *hist4 = reinterpret_cast<int64_t *>(ws);
    ws += align_up((size_t)B * 4 * 8, 256);
    const size_t a1_bytes = ensemble_a1_scratch(CB, N);
    unsigned char *a1ws = static_cast<unsigned char *>(workspace) + cs_bd_action_batched_host_workspace(B, N, dim) - a1_bytes;
    const size_t left = (size_t)(a1ws - ws);
    const int64_t kmax = clamp_kmax(N, 3);

    // the copy stream may not touch the workspace before the caller's stream is done with earlier work on it
    CS_CUDA(cudaEventRecord(start, st));
    CS_CUDA(cudaStreamWaitEvent(copy_stream, start, 0));
    int64_t c = 0;
    for (int64_t b0 = 0; b0 < B; b0 += CB, c++) {
        const int64_t nb = (B - b0 < CB) ? B - b0 : CB;
        const int buf = (int)(c & 1);
        const int rc = [&]() -> int {
            if (c >= 2) CS_CUDA(cudaStreamWaitEvent(copy_stream, consumed[buf], 0));
            CS_CUDA(cudaMemcpyAsync(cdev[buf], coords_host + b0 * N * dim, (size_t)nb * N * dim * 8,
                                    cudaMemcpyHostToDevice, copy_stream));
            CS_CUDA(cudaEventRecord(copied[buf], copy_stream));
            CS_CUDA(cudaStreamWaitEvent(st, copied[buf], 0));
            const bool fits = cs_causal_matrix_workspace(nb, N, dim, geometry, CS_A1_AUTO) <= a1_bytes;
            int r = cs_causal_matrix_ex(cdev[buf], nb, N, dim, geometry, CS_A1_AUTO, bits, bitsT, fits ? a1ws : nullptr,
                                        fits ? a1_bytes : 0, stream);
            if (r) return r;
            CS_CUDA(cudaEventRecord(consumed[buf], st));
            if (kmax < 3) CS_CUDA(cudaMemsetAsync(hist, 0, (size_t)nb * 4 * 8, st));
            r = interval_hist_impl(bits, bitsT, nb, N, kmax, 0, N, CS_ROUTE_AUTO, hist, nullptr, ws, left, st, b0 > 0);
            if (r) return r;
            return launch_bd_action(hist, kmax + 1, nb, kmax, N, spacetime_dim(geometry, dim), actions + b0, nullptr,
                                    hist4 + b0 * 4, st);
        }();
        if (rc) {   // do not hand the caller's coords_host back while the copy stream may still be reading it
            cudaStreamSynchronize(copy_stream);
            return rc;
        }
    }
    CS_CUDA(cudaMemcpyAsync(actions_host, actions, (size_t)B * 8, cudaMemcpyDeviceToHost, st));
    if (hist4_host) CS_CUDA(cudaMemcpyAsync(hist4_host, hist4, (size_t)B * 4 * 8, cudaMemcpyDeviceToHost, st));
    CS_CUDA(cudaStreamSynchronize(st));
    return CS_OK;
}

// ---- end to end with host buffers ----------------------------------------------------------
// workspace: [coords][bits][bitsT][hist][action+pad][interval scratch]
size_t cs_action_host_workspace(int64_t N, int64_t kmax)
{
    if (N < 0) return 0;
    kmax = clamp_kmax(N, kmax);
    const size_t mat = align_up((size_t)N * row_stride_words(N) * 8, 256);
    return align_up((size_t)N * 7 * 8, 256) + 2 * mat + align_up((size_t)(kmax + 1) * 8, 256) + 256 +
           interval_ws_bytes(1, N, 1, cs_default_route(N)) + ensemble_a1_scratch(1, N);
}

int cs_action_host(const double *coords_host, int64_t N, int dim, int geometry, int64_t kmax,
                   int64_t *hist_host, double *action_host,
                   void *workspace, size_t workspace_bytes, void *stream)
{
    if (N < 0 || !hist_host || !action_host || (N > 0 && !coords_host)) return CS_ERR_ARG;
    {
        const int rc = check_pipeline_args(N, dim, geometry);
        if (rc) return rc;
    }
    if (!workspace || workspace_bytes < cs_action_host_workspace(N, kmax) || ((uintptr_t)workspace & 255))
        return CS_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    kmax = clamp_kmax(N, kmax);
    const size_t mat = align_up((size_t)N * row_stride_words(N) * 8, 256);
    unsigned char *ws = static_cast<unsigned char *>(workspace);
    double *coords = reinterpret_cast<double *>(ws);
    ws += align_up((size_t)N * 7 * 8, 256);
    uint64_t *bits = reinterpret_cast<uint64_t *>(ws);
    ws += mat;
    uint64_t *bitsT = reinterpret_cast<uint64_t *>(ws);
    ws += mat;
    int64_t *hist = reinterpret_cast<int64_t *>(ws);
    ws += align_up((size_t)(kmax + 1) * 8, 256);
    double *action = reinterpret_cast<double *>(ws);
    ws += 256;
    const size_t a1_bytes = ensemble_a1_scratch(1, N);
    unsigned char *a1ws = static_cast<unsigned char *>(workspace) + cs_action_host_workspace(N, kmax) - a1_bytes;
    const size_t left = (size_t)(a1ws - ws);

    if (N > 0) CS_CUDA(cudaMemcpyAsync(coords, coords_host, (size_t)N * dim * 8, cudaMemcpyHostToDevice, st));
    const bool fits = cs_causal_matrix_workspace(1, N, dim, geometry, CS_A1_AUTO) <= a1_bytes;
    int rc = cs_causal_matrix_ex(coords, 1, N, dim, geometry, CS_A1_AUTO, bits, bitsT, fits ? a1ws : nullptr, fits ? a1_bytes : 0, stream);
    if (rc) return rc;
    rc = cs_interval_hist(bits, bitsT, N, kmax, hist, nullptr, ws, left, stream);
    if (rc) return rc;
    rc = cs_bd_action(hist, kmax, N, spacetime_dim(geometry, dim), action, nullptr, stream);
    if (rc) return rc;
    CS_CUDA(cudaMemcpyAsync(hist_host, hist, (size_t)(kmax + 1) * 8, cudaMemcpyDeviceToHost, st));
    CS_CUDA(cudaMemcpyAsync(action_host, action, 8, cudaMemcpyDeviceToHost, st));
    CS_CUDA(cudaStreamSynchronize(st));
    return CS_OK;
}

}  // extern "C"
