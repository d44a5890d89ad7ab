/*
 * causalset.h -- C ABI of libcausalset.so: the causal-set action hot path of
 * W. J. Cunningham, "High Performance Algorithms for Quantum Gravity and
 * Cosmology" (arXiv:1805.04463), hand-written CUDA for sm_100a (B200).
 *
 * Path (citations are PAPER.md line numbers; readings A1..A15 are in DESIGN.md):
 *   a1  cs_causal_matrix   coordinates -> bit-packed causal matrix
 *   a2  cs_interval_hist   bits -> interval abundances N_k           (Alg. 19/20)
 *   a3  cs_bd_action       N_k -> Benincasa-Dowker action            (Eq. 4.10-4.12)
 *
 * Conventions common to every entry point
 *   - "device" pointers are caller-owned CUDA device memory (e.g. from torch);
 *     "host" pointers are ordinary host memory.  The library never allocates
 *     or frees an output and keeps no pointer after the call returns.  One call
 *     takes scratch of its own when it is given none: cs_causal_matrix /
 *     cs_causal_matrix_batched / cs_causal_matrix_ex with workspace = NULL on the
 *     tensor route, from a stream-ordered memory pool the library owns per device
 *     (allocated and freed in stream order inside the call; the pool keeps the
 *     memory for the next call).  Pass a workspace to avoid it.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default
 *     stream).  Device-pointer calls only enqueue work and return; results are
 *     valid after the stream is synchronised.  *_host calls synchronise.
 *   - every call returns a cs_status (0 = ok, <0 = error); nothing throws.
 *     On error no output is guaranteed.  There is no CPU fallback: without a
 *     CUDA device every compute call returns CS_ERR_CUDA.
 *   - bit layout (FastBitset): a matrix is N rows
 *     of `stride = cs_row_stride_words(N)` uint64 blocks; element j of a row is
 *     bit (j & 63) of block (j >> 6), LSB first; padding bits are zero.
 *   - elements must be sorted by non-decreasing time coordinate
 *     so that i -< j implies i < j; only pairs i < j are ever tested.
 *   - threads and devices: calls may come from several host threads and for several devices of one
 *     process (the device is the calling thread's current one; everything the library caches on the host
 *     is keyed by it).  Two calls that share a workspace, or two *_host calls on the same device, must
 *     not run concurrently.
 */
#ifndef CAUSALSET_H
#define CAUSALSET_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Geometry of the sprinkled region = the pairwise predicate "i precedes j". */
enum cs_geometry {
    /* dim = 2, coords (u,v) light-cone coordinates, ds^2 = -2 du dv:
       i -< j  <=>  u_i < u_j && v_i < v_j. */
    CS_GEOM_MINK2_LIGHTCONE = 0,
    /* dim = 2..5, coords (t,x[,y[,z[,w]]]) (squared form of Eq. 7.7; dim 5 = the 4+1
       diamond of App. A.1.2):
       dt = t_j - t_i, d_a = x^a_j - x^a_i, s = (((dx*dx) + (dy*dy)) + (dz*dz)) + (dw*dw),
       i -< j  <=>  dt >= 0 && dt*dt >= s        (fp64, no FMA contraction). */
    CS_GEOM_MINK_CONE = 1,
    /* dim = 2, coords (eta,theta) of the 1+1 de Sitter slab (Eq. 4.19):
       a = |theta_j - theta_i|, b = 2pi - a, m = a < b ? a : b,
       i -< j  <=>  eta_j - eta_i >= m           (2pi = 0x401921FB54442D18). */
    CS_GEOM_DS2_SLAB = 2,
    /* dim = 6, a point is (eta, r, cos th, sin th, cos ph, sin ph): conformally flat 3+1 FLRW in conformal
       time and spherical coordinates, Eq. 7.7, strict as printed; cos(ph_i - ph_j) is
       expanded, so the trigonometric values are taken once per point by the caller:
       cphi = (cp_i*cp_j) + (sp_i*sp_j), ang = (ct_i*ct_j) + ((st_i*st_j)*cphi),
       d2 = ((r_i*r_i) + (r_j*r_j)) - ((2*(r_i*r_j))*ang), deta = eta_j - eta_i,
       i -< j  <=>  deta > 0 && d2 < deta*deta   (fp64, no FMA contraction).
       The spacetime dimension (for the action entry points that take coordinates) is 4. */
    CS_GEOM_FLRW_POLAR = 3,
    /* dim = 7, a point is (eta, cos eta, sin eta, X0, X1, X2, X3): 3+1 de Sitter with spherical foliation,
       ds^2 = lambda^2 sec^2(eta) (-d eta^2 + d Omega_3^2) (App. A.1.3), X = (cos psi,
       sin psi cos th, sin psi sin th cos ph, sin psi sin th sin ph) the point's unit vector on the 3-sphere.
       Timelike <=> d eta^2 > d Sigma^2 with d Sigma = omega the great-circle angle; for
       0 < d eta <= pi that is cos(d eta) < cos(omega) (reading A18):
       cd = (ce_i*ce_j) + (se_i*se_j), co = ((X0_i*X0_j) + (X1_i*X1_j)) + ((X2_i*X2_j) + (X3_i*X3_j)),
       i -< j  <=>  eta_j - eta_i > 0 && cd < co   (fp64, no FMA contraction; strict like Eq. 7.7).
       The spacetime dimension (for the action entry points that take coordinates) is 4. */
    CS_GEOM_DS4_SPHERICAL = 4
};

enum cs_status {
    CS_OK = 0,
    CS_ERR_ARG = -1,        /* NULL pointer, negative size, misaligned buffer */
    CS_ERR_DIM = -2,        /* dim not valid for the geometry / action */
    CS_ERR_GEOM = -3,       /* unknown geometry */
    CS_ERR_UNSORTED = -4,   /* reserved (the library does not check sortedness) */
    CS_ERR_WORKSPACE = -5,  /* workspace NULL or smaller than the *_workspace() query */
    CS_ERR_CUDA = -6,       /* a CUDA runtime call or launch failed; see cs_last_cuda_error() */
    CS_ERR_CAPACITY = -7    /* the size is beyond the fixed capacity of an entry point that owns its scratch
                               (cs_interval_hist_static); cs_last_cuda_error() names the limit */
};

/* How a2 is computed.  All routes give identical integers. */
enum cs_route {
    CS_ROUTE_AUTO = 0,      /* the library's default for this N: CS_ROUTE_TENSOR_PAIR for 1024 <= N <= 2^21 on a device that
                               passed cs_a2_tensor_selfcheck, else CS_ROUTE_POPC */
    CS_ROUTE_POPC = 1,      /* shared-memory tiled AND + POPC (Alg. 20 restated for the GPU) */
    CS_ROUTE_TENSOR = 2,    /* count matrix C.C as a 0/1 int8 contraction on tcgen05 tensor cores */
    CS_ROUTE_TENSOR_FP4 = 3,/* the same contraction with 4-bit (E2M1, unit block scales) operands, fp32 accumulators */
    CS_ROUTE_TENSOR_PAIR = 4/* 4-bit operands on CTA pairs (cta_group::2, 256 x 256 tiles), shift-free expansion with
                               constant power-of-two block scales, L2-aware tile order; K blocks whose 256 x 256 bit
                               block is empty are not executed (large single causets).  The default for N >= 1024.
                               The tensor routes assume bits is upper triangular (as cs_causal_matrix writes it). */
};

const char *cs_version(void);
const char *cs_status_string(int status);
/* Text of the last CUDA error seen by this thread's calls ("" if none). Host string, static storage. */
const char *cs_last_cuda_error(void);

/* Row stride in uint64 blocks: ceil(N/64) rounded up to an even count (rows are 128-bit aligned). */
int64_t cs_row_stride_words(int64_t N);

/* a1: causal matrix.
 *   coords  device, [N][dim] fp64, time coordinate first, sorted by time; 16-byte aligned.
 *   bits    device, [N][stride] uint64, overwritten: bit j of row i = (i < j && i -< j)
 *           (upper triangular: "future of i"); lower triangle and padding are written as zero.
 *   bitsT   device or NULL, [N][stride] uint64, overwritten with the transpose
 *           (bit i of row j = i -< j: "past of j").
 * Errors: CS_ERR_ARG (NULL coords/bits, N < 0), CS_ERR_GEOM, CS_ERR_DIM, CS_ERR_CUDA.  N = 0 is a no-op. */
int cs_causal_matrix(const double *coords, int64_t N, int dim, int geometry,
                     uint64_t *bits, uint64_t *bitsT, void *stream);

/* Same for B independent causets: coords [B][N][dim], bits/bitsT [B][N][stride]. */
int cs_causal_matrix_batched(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                             uint64_t *bits, uint64_t *bitsT, void *stream);

/* How a1 is computed.  Both routes write identical bits. */
enum cs_a1_route {
    CS_A1_AUTO = 0,         /* the library's choice for this geometry and size */
    CS_A1_FMA = 1,          /* every geometry: predicate on the FMA pipes (exact fp32 prefilter, fp64 inside its error band) */
    CS_A1_TENSOR = 2        /* the predicate as the sign of a bilinear form (every geometry has one: the 1+1 light cone as
                               du dv, the 1+1 dS slab as cos dtheta - cos d eta, the others as in CS_A1_FMA's prefilter),
                               evaluated as a split-bf16 contraction on tcgen05 tensor cores; rows of a 32 x 32 block with a
                               value inside the error band are re-evaluated with the fp64 expression.  N >= 256 (CS_ERR_ARG
                               below that). */
};

/* a1 with the route chosen by the caller and an optional workspace (B causets, B = 1 for a single one).
 *   workspace  device, >= cs_causal_matrix_workspace() bytes, 256-byte aligned, or NULL: the tensor route then takes its
 *              scratch (operand rows of the points, 128 B per point and less than 1 % of the matrices) from a
 *              stream-ordered memory pool the library owns on this device.
 * bits / bitsT must be 16-byte aligned.  Errors as cs_causal_matrix, + CS_ERR_WORKSPACE. */
size_t cs_causal_matrix_workspace(int64_t B, int64_t N, int dim, int geometry, int route);
/* What CS_A1_AUTO resolves to for B causets of N points by size alone: CS_A1_TENSOR once the launch has
 * at least 128 tiles of 256 x 256 pairs (one causet: N >= 3841; ensembles earlier; always N >= 256), else CS_A1_FMA.
 * Host logic only: it does not consult the device's self-check (cs_a1_tensor_selfcheck), so on a device that failed
 * it -- or on which the check could not run -- AUTO runs the FMA route although this call, and
 * cs_causal_matrix_workspace(route = AUTO), still answer for the tensor route (the workspace is then simply unused). */
int cs_default_a1_route(int64_t B, int64_t N, int dim, int geometry);
int cs_causal_matrix_ex(const double *coords, int64_t B, int64_t N, int dim, int geometry, int route,
                        uint64_t *bits, uint64_t *bitsT, void *workspace, size_t workspace_bytes, void *stream);

/* CS_A1_TENSOR on one flat-cone causet (dim 4 or 5) with its counters on: what the tensor-core value of the bilinear form
 * was worth on this input.  Writes bits / bitsT as cs_causal_matrix does.
 *   out_host  host, double[5], overwritten: [0] the largest |a - T| seen, in units of 2^-24 C^2 (a = tensor-core value,
 *             T = the form evaluated in fp64, C = largest |coordinate| of the tile; over all pairs decided by sign),
 *             [1] (row, 32-column block) pairs re-evaluated in fp64, [2] (row, block) pairs examined, [3] the largest
 *             |a - T| / m, m = the margin of the pair's tile (a decision by sign can only be wrong if this reaches 1),
 *             [4] the largest |a - S| in the unit of [0], S = the exact sum of the products of the bf16 operand pieces
 *             the tensor core was given (its accumulation error alone).
 * Synchronises `stream`.  Errors: CS_ERR_ARG (also N < 256), CS_ERR_DIM, CS_ERR_WORKSPACE, CS_ERR_CUDA. */
int cs_a1_tensor_probe(const double *coords, int64_t N, int dim, uint64_t *bits, uint64_t *bitsT,
                       void *workspace, size_t workspace_bytes, double *out_host, void *stream);

/* The self-check behind CS_A1_AUTO.  The tensor route's error band rests on a model of the tensor core's accumulation
 * (reading A21); the first time AUTO would take that route on a device the library runs the probe above on a
 * seeded causet of 2048 points in 3+1 and in 4+1 dimensions and keeps the FMA route on that device if the largest
 * |a - T| / m reaches 0.25.  This call runs the check if it has not run yet and reports it: 1 the device behaves like the
 * model, 0 it does not (AUTO = FMA route there; CS_A1_TENSOR by name still runs), < 0 a cs_status.  Synchronises `stream`
 * the first time (about 1 ms), then returns the cached answer. */
int cs_a1_tensor_selfcheck(void *stream);

/* bitsT <- transpose(bits) (both device, [N][stride]); for callers that kept only `bits`. */
int cs_transpose_bits(const uint64_t *bits, int64_t N, uint64_t *bitsT, void *stream);

/* Relation count R = popcount(bits) and the algorithmic work of Alg. 20,
 * W_alg = sum over related pairs of ((j>>6) - (i>>6) + 1) 64-bit blocks.
 *   out  device, int64[2] = {R, W_alg}, overwritten. */
int cs_relation_stats(const uint64_t *bits, int64_t N, int64_t *out, void *stream);

/* Degree vectors (the by-product of the paper's linker, Alg. 17):
 *   outdeg[k] = number of elements in the future of k (row sum of bits),
 *   indeg[k]  = number of elements in its past (row sum of bitsT).
 * Both device, int64[N]; either may be NULL (indeg needs bitsT).  sum_k indeg[k] outdeg[k] is the number of
 * 3-chains = sum_k k hist[k] (used as a whole-size check of a2). */
int cs_degrees(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t *outdeg, int64_t *indeg, void *stream);

/* a2: interval abundances (Alg. 19; Alg. 20).
 * For every related pair i -< j:  c = |{k : i -< k -< j}| = popcount(bits[i] & bitsT[j]);  hist[c] += 1.
 * hist[k] = n_{k+1} in the paper's notation (Eq. 4.8).
 *   bits, bitsT  device, as produced by cs_causal_matrix; 16-byte aligned (rows are read with 128-bit
 *                loads, bulk copies and TMA; CS_ERR_ARG otherwise).  bitsT may be NULL: it is then
 *                rebuilt inside the workspace (query the size with have_bitsT = 0).
 *   kmax         largest interval size kept; kmax < 0 or kmax > N-2 means N-2.
 *   hist         device, int64[kmax+1] (after clamping; at least 1 entry), overwritten.
 *                Pairs with c > kmax are dropped from hist but counted in *n_relations.
 *   n_relations  device int64[1] or NULL: number of related pairs (restricted to the row range).
 *   workspace    device, >= cs_interval_hist_workspace() bytes, 256-byte aligned; scratch.
 * cs_interval_hist_ex restricts the outer element i to [row_begin, row_end) (hist then holds
 * the contribution of those rows only: partial histograms add up) and selects the route.
 * Errors: CS_ERR_ARG, CS_ERR_WORKSPACE, CS_ERR_CUDA.  N < 2 zeroes the outputs. */
size_t cs_interval_hist_workspace(int64_t N, int64_t kmax, int have_bitsT, int route);
int cs_interval_hist(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                     int64_t *hist, int64_t *n_relations,
                     void *workspace, size_t workspace_bytes, void *stream);
int cs_interval_hist_ex(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                        int64_t row_begin, int64_t row_end, int route,
                        int64_t *hist, int64_t *n_relations,
                        void *workspace, size_t workspace_bytes, void *stream);
/* a2 for callers that cannot allocate device memory.
 *
 * Every other a2 call wants a workspace, and somebody has to cudaMalloc it.  Some callers can't: code that runs inside
 * another framework's allocator hook or while that framework's caching allocator is locked; a service whose device
 * memory is budgeted once at start-up and must not grow (real-time, embedded, multi-tenant with a hard quota); a plugin
 * that receives nothing but its input and output buffers.  This entry point is for them: the same result as
 * cs_interval_hist_ex(route = CS_ROUTE_POPC) over all rows (Alg. 20), with the scratch -- the tile
 * counter and, if bitsT is NULL, the transposed matrix -- in a static array inside the library's device image.
 * It calls no cudaMalloc, cudaFree, memory-pool or other allocating routine; the caller still owns inputs and outputs.
 *   bits, bitsT, kmax, hist, n_relations   exactly as for cs_interval_hist (bitsT may be NULL).
 *   N            at most cs_interval_hist_static_max_n() = 8192.  Larger N returns CS_ERR_CAPACITY and
 *                cs_last_cuda_error() states the limit; nothing is written.
 * Cost: the array is 8 MiB + 256 B of device memory on every GPU that loads the library, from load until exit,
 * whether or not this call is ever made.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress) and sets the kernel's
 * shared-memory attribute, once, with the calling thread's current device.  Make that first call outside any stream
 * capture, e.g. once at start-up on a tiny input.
 * Sharing: all calls on a device use the one array and it keeps what the previous call left.  The call clears what
 * has to start at zero itself (in stream order), so back-to-back calls on ONE stream are fine; two calls whose work
 * can overlap on the GPU (different streams, different host threads) race on the array and give wrong histograms --
 * serialise them.
 * Errors: CS_ERR_ARG, CS_ERR_CAPACITY, CS_ERR_CUDA.  N < 2 zeroes the outputs. */
int64_t cs_interval_hist_static_max_n(void);
int cs_interval_hist_static(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t kmax,
                            int64_t *hist, int64_t *n_relations, void *stream);

/* The self-check behind CS_ROUTE_AUTO.  CS_ROUTE_TENSOR_PAIR reads its counts out of the bit patterns of subnormal
 * fp32 accumulators, exact only while the tensor cores add subnormals without flushing or rounding them (DESIGN.md,
 * reading A22: measured, not documented by the vendor).  The first time AUTO would take that route on a device the
 * library runs it on a built-in total order of 2125 elements (closed form N_k = N-1-k, every count 0..N-2 occurs) and
 * on a seeded 3+1 causet against the POPC route (whole histogram, and kmax = 3); on any difference AUTO keeps the POPC
 * route on that device (the workspace AUTO asked for is large enough for it) and cs_last_cuda_error() says what
 * differed.  This call runs the check if it has not run yet and reports it: 1 exact, 0 not (AUTO = POPC there;
 * CS_ROUTE_TENSOR_PAIR by name still runs), < 0 a cs_status.  The first time it takes ~2 MiB from the library's
 * stream-ordered pool and synchronises `stream` (about 1 ms); then it returns the cached answer.  Neither self-check
 * runs while `stream` is being captured into a CUDA graph (it would invalidate the capture): an AUTO call made during
 * capture on a device that has not been checked yet records the POPC (a1: FMA) route into the graph, and this call then
 * reports 0 without caching it.  Call it once at start-up, outside any capture, to have the tensor routes in graphs. */
int cs_a2_tensor_selfcheck(void *stream);

/* What the last cs_interval_hist* call that used `workspace` executed (for the roofline on executed work):
 *   stats_host  host, int64[4], overwritten:
 *     [0] (tile, stage) pairs whose MMAs were issued: a stage is 256 rows x 256 columns x 256 k of the 0/1
 *         contraction = 2 * 256^3 tensor ops (CS_ROUTE_TENSOR_PAIR; 0 for the other routes),
 *     [1] the same count with no empty block skipped (the dense-triangular tile set of the row range),
 *     [2] empty 256 x 256 bit blocks found by the flag pass, [3] blocks it examined (0 if it did not run).
 * Copies 64 bytes device->host and synchronises `stream`.  Errors: CS_ERR_ARG, CS_ERR_CUDA. */
int cs_interval_hist_stats(const void *workspace, int64_t *stats_host, void *stream);

/* NEXT-3: chains and antichains on the bit matrix (Algorithms 11-13).
 * Both take bits and bitsT as written by cs_causal_matrix and a workspace of cs_poset_workspace(N) bytes
 * (256-byte aligned).
 *
 * cs_chain_heights: height[k] = number of elements of the longest chain that ends at element k (1 for a
 * minimal element).  With source >= 0 only chains starting at `source` count: height[source] = 1, 0 for
 * elements outside the future of `source`; then height[j] - 1 is the result of Algorithm 11 for the pair
 * (source, j): the number of links of the longest chain between them.  source = -1: all chains.
 *   height   device, int32[N], overwritten.
 *   longest  device, int64[1] or NULL: the largest height (0 for N = 0).
 *
 * cs_greedy_antichain: Algorithm 13 with seed element `seed`: candidates = elements unrelated to the seed;
 * repeatedly keep the candidate j that leaves the most elements, c = |A \ J(j)|, J(j) = future | past of j
 * (the first such j in index order), and drop its relatives, until no candidate is left.
 *   member   device, uint64[cs_row_stride_words(N)], overwritten: bit k set iff element k is in the antichain.
 *   size     device, int64[1] or NULL: number of members.
 * Errors: CS_ERR_ARG (source/seed out of range), CS_ERR_WORKSPACE, CS_ERR_CUDA. */
size_t cs_poset_workspace(int64_t N);
int cs_chain_heights(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t source,
                     int32_t *height, int64_t *longest, void *workspace, size_t workspace_bytes, void *stream);
int cs_greedy_antichain(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t seed,
                        uint64_t *member, int64_t *size, void *workspace, size_t workspace_bytes, void *stream);

/* a2 over B causets in one launch (the Monte-Carlo ensemble): bits/bitsT are
 * [B][N][stride] as written by cs_causal_matrix_batched (bitsT required), hist is int64[B][kmax+1]
 * (kmax clamped as above), overwritten.  Workspace: cs_interval_hist_batched_workspace() bytes.
 * Errors: CS_ERR_ARG, CS_ERR_WORKSPACE, CS_ERR_CUDA. */
size_t cs_interval_hist_batched_workspace(int64_t B, int64_t N, int route);
int cs_interval_hist_batched(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                             int route, int64_t *hist, void *workspace, size_t workspace_bytes, void *stream);
/* Route CS_ROUTE_AUTO resolves to for this N (one of the concrete routes). */
int cs_default_route(int64_t N);

/* a3: Benincasa-Dowker action, Eq. 4.10-4.12 with l/l_p = 1:
 *   dim 2: S = 2 (N - 2 N_0 + 4 N_1 - 2 N_2)
 *   dim 3: S = (1/Gamma(5/3)) (pi/(3 sqrt 2))^(2/3) (N - N_0 + (27/8) N_1 - (9/4) N_2)
 *   dim 4: S = (4/sqrt 6) (N - N_0 + 9 N_1 - 16 N_2 + 8 N_3)
 *   hist     device, int64[kmax+1]; entries beyond kmax are taken as 0.
 *   action   device, double[1], overwritten.
 *   bracket  device int64[1] or NULL: the exact integer bracket (dim 2, 4) or 8 x bracket (dim 3).
 * Errors: CS_ERR_ARG, CS_ERR_DIM, CS_ERR_CUDA. */
int cs_bd_action(const int64_t *hist, int64_t kmax, int64_t N, int dim,
                 double *action, int64_t *bracket, void *stream);

/* Smeared (non-local) action S_eps, Eq. 4.13-4.15 with the smearing functions of Eq. 4.16-4.18
 * (PAPER.md:1783-1795), l/l_p = 1, from the FULL interval histogram:
 *   dim 2: S = 2 eps [ N - 2 eps sum_k hist[k] f_2(k, eps) ]
 *   dim 3: S = (1/Gamma(5/3)) (pi eps/(3 sqrt 2))^(2/3) [ N - eps sum_k hist[k] f_3(k, eps) ]
 *   dim 4: S = 4 sqrt(eps/6) [ N - eps sum_k hist[k] f_4(k, eps) ]
 * (the paper's n_m f(m-1) with m = k+1).  f_d is evaluated in the polynomial form
 * (1-eps)^k - c1 k eps (1-eps)^(k-1) + ..., which is also defined at eps = 1, where S_eps equals the
 * local action of cs_bd_action.  The sum is carried in double-double arithmetic (it cancels to a small
 * fraction of its terms) and rounded to fp64 once at the end.
 *   hist    device, int64[kmax+1] (kmax clamped as in cs_interval_hist; entries beyond kmax count as 0,
 *           so pass the whole histogram, kmax = N-2, for the paper's S_eps).
 *   eps     0 < eps <= 1.
 *   action  device, double[1], overwritten.
 * Errors: CS_ERR_ARG (eps out of range, N > 131073), CS_ERR_DIM, CS_ERR_CUDA. */
int cs_smeared_action(const int64_t *hist, int64_t kmax, int64_t N, int dim, double eps,
                      double *action, void *stream);

/* Batched ensemble (Monte-Carlo use): B independent causets of N points each,
 * one action per causet.  The ensemble is built and reduced chunk by chunk (a whole number of causets per CTA
 * pair of a2's grid, at most 500 MiB of bit matrices and a1 scratch at a time), so the workspace does not grow with B beyond
 * 32 bytes per causet.
 *   coords   device, [B][N][dim] fp64, each causet sorted by time.
 *   actions  device, double[B], overwritten.
 *   hist4    device int64[B][4] or NULL: N_0..N_3 of every causet.
 *   workspace device, >= cs_bd_action_batched_workspace(B, N) bytes, 256-byte aligned. */
size_t cs_bd_action_batched_workspace(int64_t B, int64_t N);
int cs_bd_action_batched(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                         double *actions, int64_t *hist4,
                         void *workspace, size_t workspace_bytes, void *stream);

/* End-to-end with HOST buffers: copies coords host->device, runs a1, a2, a3, copies hist and
 * the action back, and synchronises the stream before returning.
 *   coords_host  host, [N][dim] fp64 (pinned memory makes the copy asynchronous).
 *   hist_host    host, int64[kmax+1] (after clamping), overwritten.
 *   action_host  host, double[1], overwritten.
 *   workspace    device, >= cs_action_host_workspace(N, kmax) bytes, 256-byte aligned. */
size_t cs_action_host_workspace(int64_t N, int64_t kmax);
int cs_action_host(const double *coords_host, int64_t N, int dim, int geometry, int64_t kmax,
                   int64_t *hist_host, double *action_host,
                   void *workspace, size_t workspace_bytes, void *stream);

/* The ensemble end to end with HOST buffers (the Monte-Carlo use): B causets of N points each,
 * processed in the same chunks as cs_bd_action_batched; the coordinates of the next chunk are copied on a library-owned
 * stream while `stream` builds and reduces the current one, so the PCIe time hides behind the kernels.  Copies the
 * actions (and N_0..N_3 per causet) back and synchronises `stream` before returning.
 *   coords_host   host, [B][N][dim] fp64; pinned memory is needed for the copies to overlap.
 *   actions_host  host, double[B], overwritten.
 *   hist4_host    host, int64[B][4] or NULL.
 *   workspace     device, >= cs_bd_action_batched_host_workspace(B, N, dim) bytes, 256-byte aligned.
 * Errors: CS_ERR_ARG, CS_ERR_DIM, CS_ERR_GEOM, CS_ERR_WORKSPACE, CS_ERR_CUDA. */
size_t cs_bd_action_batched_host_workspace(int64_t B, int64_t N, int dim);
int cs_bd_action_batched_host(const double *coords_host, int64_t B, int64_t N, int dim, int geometry,
                              double *actions_host, int64_t *hist4_host,
                              void *workspace, size_t workspace_bytes, void *stream);

/* Peak probes -- a measurement aid for the rooflines bench.py reports ("pipe utilisation vs the
 * measured peaks"), not a step of the path.  Each probe saturates one unit with the instruction the path's
 * kernels use on it and synchronises before returning.
 *   iters      inner iterations (MMAs for the tensor probes); clamped to [4, 2^22].
 *   workspace  device, 256-byte aligned, >= 64 KiB; the HBM probes stream over everything beyond the first
 *              64 KiB and need >= 256 MiB there (CS_ERR_WORKSPACE otherwise).
 *   out_host   host, double[3]: {units executed, seconds (CUDA events), units per clock per SM (in-kernel
 *              clock64 of the slowest CTA; 0 for the HBM probes)}.  Units: tensor probes -- operations (2 per
 *              multiply-add); POPC / DFMA / FFMA -- lane-instructions; FFMA2 -- fused multiply-adds (two per
 *              lane-instruction); HBM -- bytes (copy: read + written); TMEM_LD -- bytes. */
enum cs_peak_kind {
    CS_PEAK_MXF4_PAIR = 0,  /* tcgen05.mma.cta_group::2.kind::mxf4.block_scale M=256 N=256 K=64 (k_interval_pair's) */
    CS_PEAK_I8 = 1,         /* tcgen05.mma.cta_group::1.kind::i8 M=128 N=256 K=32 (k_interval_tensor's) */
    CS_PEAK_POPC = 2,       /* POPC.32 */
    CS_PEAK_DFMA = 3,       /* fp64 fused multiply-add */
    CS_PEAK_FFMA = 4,       /* fp32 fused multiply-add */
    CS_PEAK_FFMA2 = 5,      /* fma.rn.f32x2 */
    CS_PEAK_HBM_WRITE = 6,  /* 128-bit stores */
    CS_PEAK_HBM_COPY = 7,   /* 128-bit loads + stores */
    CS_PEAK_TMEM_LD4 = 8,   /* tcgen05.ld 32x32b.x32, one warp per TMEM lane quarter */
    CS_PEAK_TMEM_LD8 = 9,   /* the same from two warps per lane quarter */
    CS_PEAK_MXF4_PAIR_N128 = 10, /* MXF4_PAIR with N = 128, alternating between two 128-column accumulator halves */
    CS_PEAK_MXF4_PAIR_N128_DEP = 11 /* MXF4_PAIR with N = 128, all into one half: a chain of dependent accumulations */
};
int cs_peak_probe(int kind, int64_t iters, void *workspace, size_t workspace_bytes, double *out_host, void *stream);

/* Number of kernel launches issued by this library in this process so far (for bench.py's
 * `gpu_launches`). */
int64_t cs_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* CAUSALSET_H */
