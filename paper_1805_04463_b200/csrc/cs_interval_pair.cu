// cs_interval_pair.cu -- stage a2, tensor route on CTA pairs (tcgen05.mma.cta_group::2, kind::mxf4).
//
// count(i,j) = sum_k U[i][k] * L[j][k] over the K blocks between the I block and the J block
// (Fig. 4.2 caption PAPER.md:1768; Alg. 20 line 9), histogrammed over related pairs.
// Same contraction as cs_interval_fp4.cu, re-cut for the two SMs of a TPC:
//
//  * a cluster of two CTAs owns a 256 (i) x 256 (j) tile.  CTA r expands the 128 U rows
//    I*256 + r*128 .. into its TMEM (A operand) and the 128 L rows J*256 + r*128 .. into its shared
//    memory (its half of the B operand); one thread of CTA 0 issues M=256 N=256 K=64 MMAs for the
//    pair.  Per SM and per k this halves the B expansion and the B shared-memory reads of the
//    single-CTA kernel (the two tensor cores share each B half), and a third of the ALU work.
//  * expansion without shifts: with x a 32-bit slice of a bit row, x & 0x11111111, x & 0x22222222 and
//    x & 0x44444444 are already E2M1 nibbles (0.5, 1.0, 2.0 where the bit is set); only bit 3 of
//    every nibble needs a shift ((x >> 3) & 0x11111111).  Each K=64 MMA takes one nibble position
//    of eight slices, so its products are all 0.25, 1 or 4 -- levelled exactly by constant UE8M0
//    block scales kept in three TMEM regions.  k is permuted inside a 256-k stage,
//    identically for both operands, which leaves the contraction unchanged.
//  * the scales are 2^-72, 2^-73, 2^-74 (not 2^1, 2^0, 2^-1): every product is then 2^-146 = eight
//    units in the last place of a SUBNORMAL fp32, and subnormals add like integers, so the bit pattern of
//    the accumulator is the integer 8 * count -- no float-to-integer step in the epilogue (the tally of the
//    ensemble case shifts by it directly: 2 instead of 4 instructions per pair).  Exact while
//    8 * count < 2^24 (the fp32 grid stays 2^-149 up to there): count < 2^21.  Measured: the tensor cores
//    accumulate subnormals without flushing; every a2 parity test runs on this path, and CS_ROUTE_AUTO takes it on a
//    device only after the self-check of cs_selfcheck.cu (reading A22).
//  * tiles are visited in a table order (longest K first; single diagonals up to nT = 160, bands of 32 diagonals with
//    snake rows beyond, see launch_interval_pair) so that the ~74 tiles in flight share a few row panels in L2.
//
// Products are 0 or 2^-146 and the fp32 accumulators are exact for counts < 2^21.
#include <cuda.h>

#include <type_traits>

#include "cs_common.cuh"

namespace cs {

namespace {

constexpr int TM = 128;                 // A rows (i) per CTA; the pair covers 256
constexpr int TILE = 256;               // rows (i) of a tile: 128 per CTA of the pair
constexpr int KSTEP = 256;              // k per stage = 4 MMAs of K = 64
constexpr int NS = 6;                   // operand stages (B in shared memory, A in TMEM)
constexpr int GK = 2;                   // stages per staged group of bit rows
constexpr int BROW = GK * 32;           // bytes per staged bit row (TMA box inner extent, 64B swizzle)
constexpr int NB = 4;                   // bit-row buffers
constexpr int TN = 256;                 // columns (j) of a tile: one 256-column fp32 accumulator
constexpr int TNH = TN / 2;             // B rows (j) per CTA (cta_group::2 splits N over the pair)
constexpr int CW = TN / 2;              // columns drained per epilogue warp
constexpr int BITS_BYTES = (TM + TNH) * BROW;        // staged bit rows per buffer
constexpr int STAGE_BYTES = TNH * (KSTEP / 2);       // this CTA's half of B, one stage
constexpr int SMEM_FIXED = NS * STAGE_BYTES + NB * BITS_BYTES + 512;      // + 4 bytes per histogram bin
// block-scaled instruction descriptor, kind::mxf4: A = B = E2M1 (1 at bits 7 and 10), both K-major,
// N >> 3 at bit 17, scale format UE8M0 (bit 23), M >> 4 at bit 24 (M = 256 over the pair), K = 64
constexpr uint32_t IDESC = (1u << 7) | (1u << 10) | ((uint32_t)(TN >> 3) << 17) | (1u << 23) | ((uint32_t)(256 >> 4) << 24);
constexpr int HS_MAX = 16896;           // shared-memory histogram bins that fit beside the operand rings
constexpr int HS_BATCHED = 2048;        // bins when several causets share a CTA (flushed at every switch)

// five warpgroups: 0-1 epilogue (warp & 3 = TMEM lane quarter, warp >> 2 = column half), 2 A expanders,
// 3 B expanders, 4 = MMA issuer, TMA loader and two idle warps.  The epilogue keeps a whole accumulator
// row slice (128 columns) in registers, so registers are re-split by warpgroup with setmaxnreg.
constexpr int EPI_WARPS = 8, EXPA_WARP0 = 8, EXPB_WARP0 = 12, EXP_WARPS = 8, MMA_WARP = 16, LOAD_WARP = 17;
constexpr int THREADS = 20 * 32;
constexpr int SMEM_BYTES = SMEM_FIXED + HS_MAX * 4;
constexpr uint32_t SF_COL = 256;        // three 16-column regions of constant scale factors: 2^-72, 2^-73, 2^-74
constexpr uint32_t A_COL = 320;         // TMEM ring of the A operand: NS x 32 columns
static_assert(A_COL + NS * 32 <= 512, "TMEM columns");
static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// arrive on the barrier at the same shared-memory offset in CTA `cta` of the cluster.  Default
// (CTA-scope) release: what the arrival publishes is consumed by the tensor cores, for which the
// writers have already issued fence.proxy.async / tcgen05.wait::st + fence::before_thread_sync;
// a cluster-scope release compiles to MEMBAR.ALL.GPU and a cluster-scope acquire to CCTL.IVALL
// (measured: 28.3 ms instead of 20 ms at N = 65536).
__device__ __forceinline__ void mbar_arrive_cluster(uint64_t *bar, uint32_t cta)
{
    uint32_t ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(bar)), "r"(cta));
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(ra) : "memory");
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
// wait on a barrier that also receives arrivals from the peer CTA (see mbar_arrive_cluster)
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity)
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
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
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
// one lane of the (converged) warp; the same lane every time
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
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_id_x()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t num_clusters_x()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}

// shared-memory matrix descriptor: no swizzle, K-major; addresses and offsets in 16-byte units
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;   // descriptor version (Blackwell)
    return d;                 // layout_type = 0 (SWIZZLE_NONE), base_offset = 0, lbo_mode = 0
}

// D[tmem] (+)= A[tmem] . B[smem], M = 256 over the CTA pair; issued by one thread of CTA 0
__device__ __forceinline__ void mma_mxf4_pair(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc,
                                              uint32_t accum, uint32_t sfa, uint32_t sfb)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%5], [%6], p;\n"
        "}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accum), "r"(sfa), "r"(sfb)
        : "memory");
}
// the barrier at this shared-memory offset in both CTAs of the pair gets one arrival when the
// MMAs issued so far have retired
__device__ __forceinline__ void mma_commit_pair(uint64_t *bar)
{
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
            smem_u32(bar)),
        "h"((uint16_t)3)
        : "memory");
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
// 32 lanes x 32 columns -> 32 registers per thread; the caller issues tcgen05.wait::ld
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t *v)
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
// 32 lanes x 16 columns <- 16 registers per thread; the caller issues tcgen05.wait::st
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};\n" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}

// E2M1 nibbles of nibble position Q = 0, 1, 2 of a 32-bit slice (values 0.5, 1, 2 where the bit is set)
template <int Q>
__device__ __forceinline__ uint32_t nib(uint32_t x)
{
    if (Q == 0) return x & 0x11111111u;
    if (Q == 1) return x & 0x22222222u;
    return x & 0x44444444u;
}
// TMEM region of the UE8M0 block scale that levels the products of nibble position q (0.25, 1, 4, 0.25)
__device__ __forceinline__ uint32_t sf_col(int q) { return SF_COL + (q == 1 ? 16u : q == 2 ? 32u : 0u); }

// ---- tile order ---------------------------------------------------------------------------------
// Tiles (I, J = I + d), 0 <= I, I + d < nT, in bands of BANDW diagonals, longest (largest d) first;
// inside a band I-major, then d ascending.  Entry = (I << 16) | J.  nT (nT + 1) / 2 entries.
// (Square tiles only: TN = 256.  Closed forms, no loops over rows: 3.6 us at nT = 256.)
__host__ __device__ inline int64_t band_tiles(int nT, int dlo, int dhi)   // sum over d of (nT - d)
{
    const int64_t w = dhi - dlo + 1;
    return w * nT - w * (int64_t)(dlo + dhi) / 2;
}
inline int64_t pair_tiles_per_causet(int64_t N)
{
    const int64_t nT = (N + TILE - 1) / TILE;
    return nT * (nT + 1) / 2;
}

__global__ void k_pair_tile_order(int nT, int BANDW, int P, int64_t total, uint32_t *__restrict__ tab)
{
    // Final position of entry p: the clusters take entries round-robin (P per round); every odd round is reversed, so
    // that the cluster that got the longest tile of one round gets the shortest of the next (with the entries in
    // descending K length this is the boustrophedon deal: N = 16384, 64 x 64 tiles: 5.6 % -> 1.4 % spread of the clusters' work).
    auto dealt = [&](int64_t p) {
        const int64_t r = p / P, c = p - r * P;
        if (!(r & 1)) return p;
        const int64_t n = total - r * P < P ? total - r * P : P;
        return r * P + (n - 1 - c);
    };
    const int b = blockIdx.x;
    const int dhi = nT - 1 - b * BANDW;
    const int dlo = dhi - BANDW + 1 > 0 ? dhi - BANDW + 1 : 0;
    const int w = dhi - dlo + 1;
    int64_t off = 0;
    for (int bb = 0; bb < b; bb++) {
        const int h = nT - 1 - bb * BANDW;
        const int l = h - BANDW + 1 > 0 ? h - BANDW + 1 : 0;
        off += band_tiles(nT, l, h);
    }
    const int full = nT - dhi;   // rows I < full have all w diagonals inside the matrix
    for (int I = threadIdx.x; I + dlo < nT; I += blockDim.x) {
        int64_t pos;
        if (I <= full) pos = (int64_t)I * w;
        else {
            const int64_t m = I - full;   // rows full .. I-1 hold nT - dlo - I' entries each
            pos = (int64_t)full * w + m * (nT - dlo) - (int64_t)(full + I - 1) * m / 2;
        }
        // d ascending in even rows, descending in odd ones: the clusters take tiles round-robin, and a snake keeps the
        // K lengths one cluster collects from a wide band even
        const int last = (dhi < nT - 1 - I ? dhi : nT - 1 - I) - dlo;      // entries of this row - 1
        for (int d = dlo; d <= dhi && I + d < nT; d++)
            tab[dealt(off + pos + ((I & 1) ? last - (d - dlo) : (d - dlo)))] = ((uint32_t)I << 16) | (uint32_t)(I + d);
    }
}

struct Tile {
    int I, J;      // 256-row block of i, TN-column block of j
    int nstages;   // 256-k stages from the first row of I to the last column of J
    int b;         // causet
    bool skip;     // no row of the tile inside [row_begin, row_end)
    // Which stages run (see "empty K blocks"): stages [0, zA) by bit k of liveA, stages [zA, zB) all,
    // stages [zB, nstages) by bit k - zB of liveB.  Without flags zA = 0, zB = nstages.
    int zA, zB;
    uint32_t liveA, liveB;
};

// ---- empty K blocks -----------------------------------------------------------------------------
// Stage k of tile (I, J) multiplies U[rows I][cols I+k] with U[rows I+k][cols J]; if either 256 x 256 bit
// block is empty the stage adds nothing.  In a time-sorted sprinkling the blocks next to the diagonal
// are empty when relations need more separation in time than a few hundred elements span (3+1 flat cone at
// N = 65536: 96 % of the diagonal blocks, half of those 5 blocks out, none beyond 16; 13.7 % of all stages).
// flagU[I][m] = block (I, I+m) non-empty, flagT[J][m] = block (J-m, J) non-empty, m < SKIPM.
constexpr int SKIPM = 16;
constexpr int SKIP_MIN_TILES = 96;      // N > 24320: below that the flag pass (~10 us) is several % of the whole call

__global__ void __launch_bounds__(256)
k_pair_block_flags(const uint64_t *__restrict__ bits, int64_t N, int64_t stride, int nT,
                   uint8_t *__restrict__ flagU, uint8_t *__restrict__ flagT, unsigned int *__restrict__ n_empty)
{
    const int I = blockIdx.x, m = blockIdx.y, K = I + m;
    if (K >= nT) return;
    const int64_t r = (int64_t)I * TILE + threadIdx.x;
    uint64_t any = 0;
    if (r < N) {
#pragma unroll
        for (int w = 0; w < TILE / 64; w++) {
            const int64_t wi = (int64_t)K * (TILE / 64) + w;
            if (wi < stride) any |= bits[r * stride + wi];
        }
    }
    const int nz = __syncthreads_or(any != 0);
    if (threadIdx.x == 0) {
        flagU[I * SKIPM + m] = (uint8_t)(nz != 0);
        flagT[K * SKIPM + m] = (uint8_t)(nz != 0);
        if (!nz) atomicAdd(n_empty, 1u);
    }
}

// sixteen 0/1 bytes -> sixteen bits
__device__ __forceinline__ uint32_t flags_to_mask(uint4 f)
{
    return ((f.x * 0x01020408u) >> 24 & 0xFu) | ((f.y * 0x01020408u) >> 24 & 0xFu) << 4 |
           ((f.z * 0x01020408u) >> 24 & 0xFu) << 8 | ((f.w * 0x01020408u) >> 24 & 0xFu) << 12;
}

// Stage k of a tile with nstages = n runs unless its U block (head window: k < SKIPM and flagU[I][k] clear) or
// its L block (tail window: t = n-1-k < SKIPM and flagT[J][t] clear) is empty.  Evaluated once per tile into the
// zone masks of Tile with bit operations; the roles only test bits (evaluating the predicate per stage in
// the expanders, which live on 64 registers, cost 16 %).
__device__ __forceinline__ uint32_t low_mask(int x) { return x >= 32 ? 0xFFFFFFFFu : (1u << x) - 1u; }
__device__ __forceinline__ void tile_zones(Tile &tc, uint32_t head, uint32_t tail)
{
    const int n = tc.nstages;
    const uint32_t deadH = ~head & 0xFFFFu;          // bit k: stage k dead through its U block
    const uint32_t deadT = ~tail & 0xFFFFu;          // bit t: stage n-1-t dead through its L block
    if (n <= 2 * SKIPM) {                            // the windows meet: one zone over the whole tile
        // tail bit t -> stage n-1-t: reverse (bit 31-t), then down by 32-n
        uint32_t live = ~(deadH | (__brev(deadT) >> (32 - n))) & low_mask(n);
        if (live == 0) live = 1;                     // nothing to add, but the accumulator must be written
        tc.zA = tc.zB = n;
        tc.liveA = live;
        tc.liveB = 0;
    } else {
        tc.zA = SKIPM;
        tc.zB = (n - SKIPM) & ~1;                    // even, so that groups of GK = 2 stages never straddle a border
        tc.liveA = head & 0xFFFFu;
        const int D = n - 1 - tc.zB;                 // 15 or 16: stage zB + t has tail index D - t
        tc.liveB = ~(__brev(deadT) >> (31 - D)) & low_mask(D + 1);
    }
}
// Calls f(k, first, second) for every group of two stages (k even) of which at least one runs; the
// loader, the expanders and the MMA issuer all walk a tile with this, so they agree by construction.
template <typename F>
__device__ __forceinline__ void for_each_group(const Tile &tc, F f)
{
    static_assert(GK == 2 && SKIPM % GK == 0, "zone borders");
    const int n = tc.nstages;
    for (int k = 0; k < tc.zA; k += GK) {
        const uint32_t pair = (tc.liveA >> k) & 3u;     // bits at or beyond nstages are 0
        if (pair) f(k, (pair & 1u) != 0, (pair & 2u) != 0);
    }
    for (int k = tc.zA; k < tc.zB; k += GK) f(k, true, k + 1 < n);
    for (int k = tc.zB; k < n; k += GK) {
        const uint32_t pair = (tc.liveB >> (k - tc.zB)) & 3u;
        if (pair) f(k, (pair & 1u) != 0, (pair & 2u) != 0);
    }
}

// SMALL: kmax <= 3 (the Monte-Carlo case, only N_0..N_3 enter Eq. 4.10-4.12): the tally keeps packed
// counters in registers and never touches the shared histogram (hs = 0).
template <bool SMALL>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
k_interval_pair(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapL,
                const uint64_t *__restrict__ bits, const uint32_t *__restrict__ tile_tab,
                const uint8_t *__restrict__ flagU, const uint8_t *__restrict__ flagT,
                const unsigned int *__restrict__ n_empty, int nT_flags, uint32_t tiles_per,
                int64_t B, int64_t N, int64_t stride, int64_t kmax, int hs, int causet_major,
                int64_t row_begin, int64_t row_end,
                unsigned long long *__restrict__ hist, unsigned long long *__restrict__ nrel,
                IntervalStats *__restrict__ stats, unsigned long long stages_total, unsigned long long blocks_examined)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *s_stage = smem;
    unsigned char *s_bits = smem + NS * STAGE_BYTES;
    uint64_t *s_full = reinterpret_cast<uint64_t *>(smem + NS * STAGE_BYTES + NB * BITS_BYTES);
    uint64_t *s_empty = s_full + NS;      // [NS] stage free again (multicast commit from CTA 0)
    uint64_t *s_tfull = s_empty + NS;     // [1 of 2 slots] accumulator complete (multicast commit)
    uint64_t *s_tempty = s_tfull + 2;     // [1 of 2 slots] accumulator drained (used in CTA 0 only)
    uint64_t *s_bfull = s_tempty + 2;     // [NB] staged bit rows have landed
    uint64_t *s_bempty = s_bfull + NB;    // [NB] every expander warp is done with the buffer
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(s_bempty + NB);
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(smem + SMEM_FIXED);   // [hs], sized by the launcher

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_ctarank();
    // 32-bit schedule state (the launcher rejects more than 2^31 tiles): the expander and issuer
    // warps run on 64 and 40 registers
    const uint32_t t0 = cluster_id_x(), tstep = num_clusters_x();
    const int ib0 = (int)(row_begin / TILE), ib1 = (int)((row_end + TILE - 1) / TILE);   // I blocks inside the row range
    const int64_t hist_len = kmax + 1;

    // Every role of both CTAs walks the same static schedule, kept as (causet, tile index) and advanced
    // without divisions.  Interleaved (one causet, or few): cluster c takes tiles c, c + #clusters, ... of the
    // concatenated tile lists.  Causet-major (ensembles): cluster c takes whole causets c, c + #clusters, ...,
    // so that the per-causet tallies are flushed once per causet, not once per tile (the ncu source view of
    // the 4096 x 2048 ensemble had two thirds of the epilogue's samples in that flush).
    struct Sched { uint32_t b, idx; };
    auto sched_first = [&]() {
        Sched sc;
        if (causet_major) { sc.b = t0; sc.idx = 0; }
        else { sc.b = t0 / tiles_per; sc.idx = t0 % tiles_per; }
        return sc;
    };
    auto sched_next = [&](Sched &sc) {
        if (causet_major) {
            if (++sc.idx == tiles_per) { sc.idx = 0; sc.b += tstep; }
        } else {
            sc.idx += tstep;
            while (sc.idx >= tiles_per) { sc.idx -= tiles_per; sc.b++; }
        }
    };
    // Testing stages costs a little even when nothing is empty (dS, 1+1 light cone): the flags are used only
    // if at least 2 % of the examined blocks turned out empty (counted by k_pair_block_flags).
    const bool use_flags = flagU != nullptr && (uint64_t)__ldg(n_empty) * 50 >= (uint64_t)nT_flags * SKIPM;
    auto get_tile = [&](const Sched &sc, bool with_zones = true) {
        Tile tc;
        tc.b = (int)sc.b;
        const uint32_t e = __ldg(tile_tab + sc.idx);
        tc.I = (int)(e >> 16);
        tc.J = (int)(e & 0xFFFFu);
        tc.nstages = ((tc.J + 1) * TN - tc.I * TILE + KSTEP - 1) / KSTEP;
        tc.skip = tc.I < ib0 || tc.I >= ib1;
        tc.zA = 0;
        tc.zB = tc.nstages;
        tc.liveA = tc.liveB = 0;
        if (with_zones && use_flags)
            tile_zones(tc, flags_to_mask(__ldg(reinterpret_cast<const uint4 *>(flagU + tc.I * SKIPM))),
                       flags_to_mask(__ldg(reinterpret_cast<const uint4 *>(flagT + tc.J * SKIPM))));
        return tc;
    };

    if (tid == 0) {
        for (int s = 0; s < NS; s++) {
            mbar_init(&s_full[s], 2 * EXP_WARPS);   // expander warps of both CTAs (counted in CTA 0)
            mbar_init(&s_empty[s], 1);
        }
        for (int b = 0; b < NB; b++) {
            mbar_init(&s_bfull[b], 1);
            mbar_init(&s_bempty[b], EXP_WARPS);
        }
        for (int a = 0; a < 2; a++) {
            mbar_init(&s_tfull[a], 1);
            mbar_init(&s_tempty[a], 2 * EPI_WARPS);     // epilogue warps of both CTAs (counted in CTA 0)
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int b = tid; b < hs; b += THREADS) s_hist[b] = 0;
    if (warp == MMA_WARP) {   // all 512 TMEM columns of both SMs of the pair
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(s_tmem)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync();           // barriers of the peer are initialised before anyone arrives on them
    tc_fence_after();
    const uint32_t tmem_base = *s_tmem;
    if (warp < 4) {           // constant UE8M0 block scales, one value in every byte of its region
        const uint32_t sf = tmem_base + ((uint32_t)(warp * 32) << 16) + SF_COL;
        tmem_st16_const(sf, 0x37373737u);          // 2^-72, 2^-73, 2^-74 on both operands
        tmem_st16_const(sf + 16, 0x36363636u);
        tmem_st16_const(sf + 32, 0x35353535u);
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync();
    tc_fence_after();

    // every role of both CTAs walks the same static schedule: tile t = cluster id, + number of clusters, ...
    // 640 threads x 96 registers at launch = the CTA's pool (setmaxnreg.inc only draws on what the CTA's
    // own warps released): 256 x 152 (epilogue) + 256 x 64 (expanders) + 128 x 40 = 61440.  Each
    // setmaxnreg sits inside its role's branch: ptxas budgets a region by the setmaxnreg that dominates it.
    if (warp >= EXPA_WARP0 && warp < MMA_WARP) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        // ===================================== expanders =====================================
        // warpgroup 2 owns this CTA's 128 A rows (row = TMEM lane: warp w may only touch lanes
        // 32 (w % 4) ..), warpgroup 3 its 128 B rows.  One thread per row.
        const bool isA = warp < EXPB_WARP0;
        const int r = (warp & 3) * 32 + lane;
        // TMA 64B swizzle: 16-byte chunk c of row e sits at chunk c ^ ((e >> 1) & 3)
        const unsigned char *my_bits = s_bits + (isA ? 0 : TM * BROW) + r * BROW;
        const int swz = (r >> 1) & 3;
        const int off0 = (0 ^ swz) << 4, off1 = (1 ^ swz) << 4, off2 = (2 ^ swz) << 4, off3 = (3 ^ swz) << 4;
        // bit 3 of every nibble is the only one that needs a shift
        auto nib3 = [&](uint32_t x) { return (x >> 3) & 0x11111111u; };
        uint32_t s = 0, ph = 0;    // operand ring position and phase
        uint32_t b = 0, bph = 0;   // bit-buffer ring position and phase
        const uint32_t a_taddr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + A_COL;
        unsigned char *b_dst = s_stage + r * 16;

        // A stage is published (arrival on its full barrier) once its stores have landed: TMEM stores
        // need tcgen05.wait::st, shared-memory stores a generic->async proxy fence.  (Deferring the wait until
        // the next stage has been expanded was measured: no difference, 10.974 vs 10.977 ms at N = 65536.)
        auto publish = [&](uint32_t stage) {
            if (isA) {
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                tc_fence_before();
            } else {
                fence_proxy_async();   // generic-proxy stores -> visible to the tensor cores
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(&s_full[stage], 0);    // one arrival per warp, in CTA 0
        };
        auto stage_A = [&](const uint4 &c0, const uint4 &c1) {
            const uint32_t xs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
            // TMEM column 8 q + j of stage s = nibble position q of slice j; two 16-column stores
            uint32_t lo[16], hi[16];
#pragma unroll
            for (int j = 0; j < 8; j++) {
                lo[j] = nib<0>(xs[j]);
                lo[8 + j] = nib<1>(xs[j]);
            }
            mbar_wait(&s_empty[s], ph ^ 1);
            tc_fence_after();
            tmem_st16(a_taddr + s * 32, lo);
#pragma unroll
            for (int j = 0; j < 8; j++) {
                hi[j] = nib<2>(xs[j]);
                hi[8 + j] = nib3(xs[j]);
            }
            tmem_st16(a_taddr + s * 32 + 16, hi);
            publish(s);
            if (++s == NS) { s = 0; ph ^= 1; }
        };
        auto stage_B = [&](const uint4 &c0, const uint4 &c1) {
            const uint32_t xs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
            uint4 w[8];       // 16-byte chunk 2 q + h of this row = nibble position q of slices 4 h .. 4 h + 3
#pragma unroll
            for (int h = 0; h < 2; h++) {
                w[0 + h] = make_uint4(nib<0>(xs[4 * h]), nib<0>(xs[4 * h + 1]), nib<0>(xs[4 * h + 2]), nib<0>(xs[4 * h + 3]));
                w[2 + h] = make_uint4(nib<1>(xs[4 * h]), nib<1>(xs[4 * h + 1]), nib<1>(xs[4 * h + 2]), nib<1>(xs[4 * h + 3]));
                w[4 + h] = make_uint4(nib<2>(xs[4 * h]), nib<2>(xs[4 * h + 1]), nib<2>(xs[4 * h + 2]), nib<2>(xs[4 * h + 3]));
                w[6 + h] = make_uint4(nib3(xs[4 * h]), nib3(xs[4 * h + 1]), nib3(xs[4 * h + 2]), nib3(xs[4 * h + 3]));
            }
            mbar_wait(&s_empty[s], ph ^ 1);
            unsigned char *dst = b_dst + s * STAGE_BYTES;
#pragma unroll
            for (int q = 0; q < 8; q++)
                *reinterpret_cast<uint4 *>(dst + q * TNH * 16) = w[q];
            publish(s);
            if (++s == NS) { s = 0; ph ^= 1; }
        };

        for (Sched sc = sched_first(); sc.b < (uint32_t)B; sched_next(sc)) {
            const Tile tc = get_tile(sc);
            if (tc.skip) continue;
            auto do_group = [&](bool first, bool second) {
                mbar_wait(&s_bfull[b], bph);
                const unsigned char *src = my_bits + b * BITS_BYTES;
                if (isA) {
                    if (first) stage_A(*reinterpret_cast<const uint4 *>(src + off0), *reinterpret_cast<const uint4 *>(src + off1));
                    if (second) stage_A(*reinterpret_cast<const uint4 *>(src + off2), *reinterpret_cast<const uint4 *>(src + off3));
                } else {
                    if (first) stage_B(*reinterpret_cast<const uint4 *>(src + off0), *reinterpret_cast<const uint4 *>(src + off1));
                    if (second) stage_B(*reinterpret_cast<const uint4 *>(src + off2), *reinterpret_cast<const uint4 *>(src + off3));
                }
                // the buffer has been loaded AND consumed by every lane (the stores above depend on
                // it): hand it back to the loader
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_bempty[b]);
                if (++b == NB) { b = 0; bph ^= 1; }
            };
            for_each_group(tc, [&](int, bool first, bool second) { do_group(first, second); });
        }
    } else if (warp >= MMA_WARP) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == LOAD_WARP && lane == 0) {
            // ===================================== TMA loader ====================================
            {
            uint32_t grp = 0;
            for (Sched sc = sched_first(); sc.b < (uint32_t)B; sched_next(sc)) {
                const Tile tc = get_tile(sc);
                if (tc.skip) continue;
                for_each_group(tc, [&](int k, bool, bool) {
                    const int b = grp % NB;
                    mbar_wait(&s_bempty[b], ((grp / NB) & 1) ^ 1);
                    mbar_arrive_expect_tx(&s_bfull[b], (uint32_t)BITS_BYTES);   // out-of-bounds is zero-filled
                    unsigned char *dst = s_bits + b * BITS_BYTES;
                    const int c0 = (tc.I * (KSTEP / 8)) + (k / GK) * BROW;      // byte column of the first k
                    tma_load_3d(dst, &mapU, c0, tc.I * TILE + (int)rank * TM, tc.b, &s_bfull[b]);
                    tma_load_3d(dst + TM * BROW, &mapL, c0, tc.J * TN + (int)rank * TNH, tc.b, &s_bfull[b]);
                    grp++;
                });
            }
        }
        } else if (warp == MMA_WARP && rank == 0) {
            // ===================================== MMA issuer (CTA 0 only) =======================
            // The whole warp walks the schedule and polls the barriers; one elected lane issues.  Kept
            // warp-uniform on purpose: with the loop inside an `if (lane == 0)` ptxas holds every MMA
            // operand in vector registers and spends ~19 instructions (R2UR, ELECT, PLOP3 ...) per MMA,
            // ~600 clk per 512-clk stage for the one issuing thread -- the kernel was bound by that
            // (ncu source view).  The shared-memory descriptor of (stage, k-slice) is the stage-0 one plus a
            // constant: the start-address field never carries out of its 14 bits (addresses < 2^18).
            const uint64_t bdesc0 = make_desc(smem_u32(s_stage), TNH * 16, 128);
            const uint32_t a_tmem0 = tmem_base + A_COL;
            const uint32_t sf0 = tmem_base + sf_col(0), sf1 = tmem_base + sf_col(1), sf2 = tmem_base + sf_col(2);
            uint32_t s = 0, ph = 0, tile_seq = 0;
            unsigned long long issued = 0;      // stages this pair executed (for cs_interval_hist_stats)
            for (Sched sc = sched_first(); sc.b < (uint32_t)B; sched_next(sc)) {
                const Tile tc = get_tile(sc);
                if (tc.skip) continue;
                mbar_wait_cluster(&s_tempty[0], (tile_seq & 1) ^ 1);      // both epilogues have drained the accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base;
                uint32_t accum = 0;                                       // the first stage that runs overwrites
                auto issue_stage = [&]() {
                    mbar_wait_cluster(&s_full[s], ph);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint64_t bd = bdesc0 + (uint64_t)((s * STAGE_BYTES) >> 4);
                        const uint32_t at = a_tmem0 + s * 32;
                        // K = 64 per MMA: 8 TMEM columns of A, 2 chunks of B
                        mma_mxf4_pair(d_tmem, at, bd, IDESC, accum, sf0, sf0);
                        mma_mxf4_pair(d_tmem, at + 8, bd + ((2 * TNH * 16) >> 4), IDESC, 1u, sf1, sf1);
                        mma_mxf4_pair(d_tmem, at + 16, bd + ((4 * TNH * 16) >> 4), IDESC, 1u, sf2, sf2);
                        mma_mxf4_pair(d_tmem, at + 24, bd + ((6 * TNH * 16) >> 4), IDESC, 1u, sf0, sf0);
                        mma_commit_pair(&s_empty[s]);                     // stage s free in both CTAs once these MMAs retire
                    }
                    __syncwarp();
                    accum = 1;
                    issued++;
                    if (++s == NS) { s = 0; ph ^= 1; }
                };
                for_each_group(tc, [&](int, bool first, bool second) {
                    if (first) issue_stage();
                    if (second) issue_stage();
                });
                if (elect_one()) mma_commit_pair(&s_tfull[0]);            // accumulator complete, both CTAs
                __syncwarp();
                tile_seq++;
            }
            if (lane == 0) {
                if (issued) atomicAdd(&stats->stages_executed, issued);
                if (t0 == 0) {
                    stats->stages_total = stages_total;
                    stats->blocks_examined = blocks_examined;
                    stats->blocks_empty = flagU ? (unsigned long long)__ldg(n_empty) : 0ull;
                }
            }
        }
    } else {
        // ===================================== epilogue ======================================
        // This CTA's accumulator: rows I*256 + rank*128 + TMEM lane, columns J*256 ...  A warp drains its
        // 32 lanes x 128 columns into registers, hands the accumulator back to the MMA issuer at
        // once, and only then tallies the related pairs -- while the next tile's MMAs run.
        asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
        uint32_t tile_seq = 0;
        unsigned long long my_nrel = 0;
        int cur_batch = -1;
        const int quarter = warp & 3, colhalf = warp >> 2;   // TMEM lane quarter; which CW = TN/2 columns
        const uint32_t taddr0 = tmem_base + ((uint32_t)(quarter * 32) << 16) + colhalf * CW;
        // The accumulator's bit pattern is 8 * count (subnormal fp32, see the header).
        const uint32_t kmax32 = (uint32_t)kmax;
        uint32_t small[4] = {0, 0, 0, 0};                    // SMALL: this thread's tallies of counts 0..3
        auto flush_small = [&](int batch) {                  // one warp reduction, <= 4 global atomics per warp
#pragma unroll
            for (int q = 0; q < 4; q++) {
                uint32_t c = small[q];
#pragma unroll
                for (int sft = 16; sft >= 1; sft >>= 1) c += __shfl_xor_sync(0xffffffffu, c, sft);
                if (lane == 0 && c && q <= kmax) atomicAdd(&hist[(int64_t)batch * hist_len + q], (unsigned long long)c);
                small[q] = 0;
            }
        };
        for (Sched sc = sched_first(); sc.b < (uint32_t)B; sched_next(sc)) {
            const Tile tc = get_tile(sc, false);
            if (tc.skip) continue;
            if (tc.b != cur_batch) {   // per-causet histograms: flush before switching
                if (cur_batch >= 0 && B > 1) {
                    if (SMALL) flush_small(cur_batch);
                    else {
                        asm volatile("bar.sync 1, 256;" ::: "memory");
                        for (int b = tid; b < hs; b += EPI_WARPS * 32) {
                            uint32_t v = s_hist[b];
                            if (v) { atomicAdd(&hist[(int64_t)cur_batch * hist_len + b], (unsigned long long)v); s_hist[b] = 0; }
                        }
                        asm volatile("bar.sync 1, 256;" ::: "memory");
                    }
                }
                cur_batch = tc.b;
            }
            const int64_t i = (int64_t)tc.I * TILE + rank * TM + quarter * 32 + lane;   // this thread's row
            const bool row_ok = i < N && i >= row_begin && i < row_end;
            uint64_t rel[2] = {0, 0};                            // relation bits of this warp's CW columns
            if (row_ok) {
                const uint64_t *urow = bits + ((int64_t)tc.b * N + i) * stride;
#pragma unroll
                for (int w = 0; w < CW / 64; w++) {
                    const int64_t wi = ((int64_t)tc.J * TN + colhalf * CW) / 64 + w;
                    if (wi < stride) rel[w] = __ldg(urow + wi);
                }
            }
            unsigned long long *ghist = hist + (int64_t)cur_batch * hist_len;
            uint32_t v[CW];
            const uint32_t taddr = taddr0;
            mbar_wait(&s_tfull[0], tile_seq & 1);
            tc_fence_after();
#pragma unroll
            for (int c = 0; c < CW / 32; c++) tmem_ld32(taddr + c * 32, &v[c * 32]);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(&s_tempty[0], 0);     // one arrival per warp, in CTA 0
            tile_seq++;
            my_nrel += __popcll(rel[0]) + __popcll(rel[1]);
            // Tally over the 128 columns in registers; 32 columns at a time are skipped when no lane of
            // the warp has a related pair there.  SMALL is branch-free (a branch per related pair
            // serialises on the latency of every step with two warps per scheduler: measured 7x the MMA
            // time of a 2048-point causet).  The general path needs one branch per column -- ptxas never
            // predicates an atomic -- and a second one only in tiles long enough to hold counts >= hs.
            uint32_t acc0 = 0, acc1 = 0;                         // SMALL: four 8-bit fields, <= 64 increments each
            const bool maybe_big = (uint32_t)tc.nstages * KSTEP > (uint32_t)hs;   // counts < 256 nstages
            auto tally = [&](auto big_tag) {
                constexpr bool BIG = decltype(big_tag)::value;
#pragma unroll
                for (int w = 0; w < CW / 32; w++) {
                    const uint32_t relw = (uint32_t)(rel[w >> 1] >> (32 * (w & 1)));
                    if (!__any_sync(0xffffffffu, relw != 0)) continue;
#pragma unroll
                    for (int c = 0; c < 32; c++) {
                        const uint32_t raw = v[w * 32 + c];                         // 8 count (see the block scales)
                        if (SMALL) {
                            // inc = 1 << 8 count; shl.b32 clamps the shift amount, so counts >= 4 give 0.
                            // SHF, predicated IADD, and one R2P per 7 columns.
                            uint32_t &acc = (c & 1) ? acc1 : acc0;
                            asm("{\n"
                                ".reg .pred r;\n"
                                ".reg .u32 t, i;\n"
                                "and.b32 t, %1, %2;\n"
                                "setp.ne.u32 r, t, 0;\n"
                                "shl.b32 i, 1, %3;\n"
                                "@r add.u32 %0, %0, i;\n"
                                "}\n" : "+r"(acc) : "r"(relw), "r"(1u << c), "r"(raw));
                        } else if (relw & (1u << c)) {
                            const uint32_t cnt = raw >> 3;
                            if (!BIG || cnt < (uint32_t)hs) atomicAdd(&s_hist[cnt], 1u);
                            else if (cnt <= kmax32) atomicAdd(&ghist[cnt], 1ULL);
                        }
                    }
                }
            };
            if (!SMALL && maybe_big) tally(std::true_type{});
            else tally(std::false_type{});
            if (SMALL) {
#pragma unroll
                for (int q = 0; q < 4; q++) small[q] += ((acc0 >> (8 * q)) & 0xFFu) + ((acc1 >> (8 * q)) & 0xFFu);
            }
        }
        // final flush by the epilogue warps
        if (SMALL) {
            if (cur_batch >= 0) flush_small(cur_batch);
        } else {
            asm volatile("bar.sync 1, 256;" ::: "memory");
            if (cur_batch >= 0) {
                for (int b = tid; b < hs; b += EPI_WARPS * 32) {
                    uint32_t v = s_hist[b];
                    if (v) atomicAdd(&hist[(int64_t)cur_batch * hist_len + b], (unsigned long long)v);
                }
            }
        }
        if (nrel && B == 1) {
#pragma unroll
            for (int s = 16; s >= 1; s >>= 1) my_nrel += __shfl_xor_sync(0xffffffffu, my_nrel, s);
            if (lane == 0 && my_nrel) atomicAdd(nrel, my_nrel);
        }
    }

    // neither CTA may leave (or free its TMEM) while the peer can still reach it
    tc_fence_before();
    __syncthreads();
    cluster_sync();
    if (warp == MMA_WARP) {
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base));
    }
}

}  // namespace

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn pair_encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// bit matrix [B][N][stride uint64] seen as bytes: dims {stride*8, N, B}; box {box_bytes, rows, 1}; 64-byte swizzle (the
// staged rows of this kernel) or none (the zero tiles cs_build_tc.cu stores)
int bits_tensor_map(CUtensorMap *map, const uint64_t *base, int64_t B, int64_t N, int64_t stride, int box_bytes, int rows,
                    bool swizzle64)
{
    EncodeTiledFn fn = pair_encode_fn();
    if (!fn) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled entry point not available");
        return CS_ERR_CUDA;
    }
    cuuint64_t gdim[3] = {(cuuint64_t)(stride * 8), (cuuint64_t)N, (cuuint64_t)B};
    cuuint64_t gstr[2] = {(cuuint64_t)(stride * 8), (cuuint64_t)(N * stride * 8)};
    cuuint32_t box[3] = {(cuuint32_t)box_bytes, (cuuint32_t)rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<uint64_t *>(base), gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed (%d)", (int)r);
        return CS_ERR_CUDA;
    }
    return CS_OK;
}
static int pair_bits_map(CUtensorMap *map, const uint64_t *base, int64_t B, int64_t N, int64_t stride, int rows)
{
    return bits_tensor_map(map, base, B, N, stride, BROW, rows, true);
}

// One 256-column accumulator per tile.  Measured alternatives that were dropped: 128-column
// tiles with two ping-pong accumulators (round 1: every A stage expanded for half the MMA work, slower at every
// size); the 256-column tile issued as two independently committed 128-column halves, the right half trailing the
// left by 1-4 stages so that one half drains while the other's MMAs run (round 2, three issuer designs, all bit-exact:
// N = 128 MMAs do run at the pipe's full rate, but holding every operand stage for the trailing half shortens the
// expanders' run-ahead and the tile is not bound by the hand-over chain but by the expanders: 10.3-10.7 ms against
// 9.8 ms at N = 65536, 0.83 against 0.80 ms per 1024 causets of N = 2048).
size_t interval_pair_scratch_bytes(int64_t N)
{
    const int64_t nT = (N + TILE - 1) / TILE;
    return align_up((size_t)pair_tiles_per_causet(N) * sizeof(uint32_t), 256) + 2 * align_up((size_t)nT * SKIPM, 256) + 256;
}

template <bool SMALL>
static int launch_pair_t(const CUtensorMap &mapU, const CUtensorMap &mapL, const uint64_t *bits, const uint32_t *tab,
                         const uint8_t *flagU, const uint8_t *flagT, const unsigned int *n_empty, int nT, uint32_t tiles_per, int64_t clusters, int64_t B, int64_t N, int64_t stride, int64_t kmax, int hs,
                         int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                         IntervalStats *stats, unsigned long long stages_total, unsigned long long blocks_examined, cudaStream_t st)
{
    static PerDeviceFlag attr_set;
    const int dev = current_device();
    if (!attr_set.get(dev)) {
        CS_CUDA(cudaFuncSetAttribute(k_interval_pair<SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     SMEM_FIXED + (SMALL ? 0 : HS_MAX * 4)));
        attr_set.set(dev);
    }
    // whole causets per cluster only if the last round of causets leaves at most 5 % of the clusters idle
    const int64_t rounds = (B + clusters - 1) / clusters;
    const int causet_major = (B > 1 && rounds * clusters * 20 <= B * 21) ? 1 : 0;
    k_interval_pair<SMALL><<<(unsigned)(2 * clusters), THREADS, SMEM_FIXED + hs * 4, st>>>(
        mapU, mapL, bits, tab, flagU, flagT, n_empty, nT, tiles_per, B, N, stride, kmax, hs, causet_major, row_begin, row_end,
        reinterpret_cast<unsigned long long *>(hist), reinterpret_cast<unsigned long long *>(nrel),
        stats, stages_total, blocks_examined);
    CS_LAUNCHED("k_interval_pair");
    return CS_OK;
}

int launch_interval_pair(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                         int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                         void *scratch, size_t scratch_bytes, IntervalStats *stats, bool keep_table, cudaStream_t st)
{
    if (N > ((int64_t)1 << 21)) return CS_ERR_ARG;   // 8 * count must stay below 2^24; tile ids are 16 bits
    static_assert(TN == TILE, "the tile table lists square tiles");
    const int64_t tiles_per = pair_tiles_per_causet(N);
    if (B > 0 && tiles_per > (((int64_t)1 << 31) - 1) / B) return CS_ERR_ARG;   // 32-bit tile schedule
    if (!scratch || scratch_bytes < interval_pair_scratch_bytes(N)) return CS_ERR_WORKSPACE;
    const int64_t stride = row_stride_words(N);
    CUtensorMap mapU, mapL;
    int rc = pair_bits_map(&mapU, bits, B, N, stride, TM);
    if (rc) return rc;
    rc = pair_bits_map(&mapL, bitsT, B, N, stride, TN / 2);
    if (rc) return rc;
    const int nT = (int)((N + TILE - 1) / TILE);
    uint32_t *tab = static_cast<uint32_t *>(scratch);
    // Band width of the tile order, from a measured sweep on B200 (a2 time / DRAM bytes read per launch).  Wide bands let the
    // ~74 tiles in flight share their row panels in L2:
    //   N = 65536 (2 x 512 MiB):  2: 9.74 ms / 23.3 GB   8: 9.81 / 9.7   16: 9.83 / 4.0   32: 9.85 / 2.3   64: 9.85 / 4.1   96: 9.91 / 7.6
    //   N = 131072 (2 x 2 GiB, power-capped at narrow bands):  2: 96.4 ms   8: 90-92 / 185 GB   16: 85.8 / 102   32: 85.8 / 84   64: 87.7 / 111
    //   N = 32768 (2 x 128 MiB): 0.3 GB at any width, 1.368 ms at 2 against 1.386 at 32
    // 32 diagonals once the matrices are well beyond L2 (1 % slower than 2 at N = 65536, but a tenth of the DRAM traffic:
    // 2.1 x the two matrices); single diagonals below (strictly descending K length, for the deal of k_pair_tile_order).
    const int bandw = nT <= 160 ? 1 : 32;
    int deal_clusters = sm_count() / 2;       // as the grid below, unless there are fewer tiles than clusters
    if (deal_clusters < 1) deal_clusters = 1;
    if (!keep_table) {
        k_pair_tile_order<<<(nT + bandw - 1) / bandw, 128, 0, st>>>(nT, bandw, deal_clusters, tiles_per, tab);
        CS_LAUNCHED("k_pair_tile_order");
    }
    // empty-block flags: one causet, and large enough that the ~10 us of the flag pass cannot matter
    uint8_t *flagU = nullptr, *flagT = nullptr;
    unsigned int *n_empty = nullptr;
    unsigned long long blocks_examined = 0;
    if (B == 1 && nT >= SKIP_MIN_TILES) {
        for (int m = 0; m < SKIPM && m < nT; m++) blocks_examined += (unsigned long long)(nT - m);
        flagU = static_cast<uint8_t *>(scratch) + align_up((size_t)tiles_per * sizeof(uint32_t), 256);
        flagT = flagU + align_up((size_t)nT * SKIPM, 256);
        n_empty = reinterpret_cast<unsigned int *>(flagT + align_up((size_t)nT * SKIPM, 256));
        CS_CUDA(cudaMemsetAsync(flagU, 0, 2 * align_up((size_t)nT * SKIPM, 256) + 256, st));   // entries no block maps to, counter
        k_pair_block_flags<<<dim3(nT, SKIPM), 256, 0, st>>>(bits, N, stride, nT, flagU, flagT, n_empty);
        CS_LAUNCHED("k_pair_block_flags");
    }
    // stages of the tiles whose rows intersect [row_begin, row_end), nothing skipped: tile (I, I+d) has d+1
    unsigned long long stages_total = 0;
    for (int64_t I = row_begin / TILE; I < (row_end + TILE - 1) / TILE && I < nT; I++)
        stages_total += (unsigned long long)((nT - I) * (nT - I + 1) / 2);
    stages_total *= (unsigned long long)B;
    const int64_t total = tiles_per * B;
    int64_t clusters = sm_count() / 2;
    if (clusters > total) clusters = total;
    if (clusters < 1) clusters = 1;
    // shared histogram: every bin up to kmax if it fits (N <= 16384 then needs no global atomics at all)
    const bool small = kmax <= 3;
    const int64_t hs_cap = B > 1 ? HS_BATCHED : HS_MAX;
    const int hs = small ? 0 : (int)(kmax + 1 < hs_cap ? kmax + 1 : hs_cap);
#define CS_PAIR_LAUNCH(S) \
    launch_pair_t<S>(mapU, mapL, bits, tab, flagU, flagT, n_empty, nT, (uint32_t)tiles_per, clusters, B, N, stride, kmax, hs, row_begin, row_end, hist, nrel, stats, stages_total, blocks_examined, st)
    return small ? CS_PAIR_LAUNCH(true) : CS_PAIR_LAUNCH(false);
#undef CS_PAIR_LAUNCH
}

}  // namespace cs
