// cs_interval_tensor.cu -- stage a2, tensor route: the count matrix C = U . U as a genuine dense
// 0/1 contraction on the 5th-generation tensor cores (tcgen05.mma kind::i8, accumulators in TMEM).
//
//   count(i,j) = |{k : i -< k -< j}| = sum_k U[i][k] * L[j][k],   U = bits ("future of i"),
//                                                                  L = bitsT ("past of j"),
// which is exactly the paper's inner product of rows i and j between columns i and j
// (Fig. 4.2 caption PAPER.md:1768; Alg. 20 line 9) with AND/popcount replaced by an
// integer multiply-accumulate.  Only K blocks between the I block and the J block are visited.
//
// Operands never exist as bytes in HBM: the bit rows are read from global memory (16 bytes = 128
// k per row per k-step) and expanded in registers straight into the shared-memory layout the MMA
// reads (no-swizzle K-major canonical layout: [16-byte k chunk][row][16 B]; SBO = 128 B,
// LBO = rows*16 B).  A bit becomes the byte 0x80 (u8 128): with x a 32-bit slice of the row,
// output word m = (x << (7-m)) & 0x80808080, i.e. byte p = 4m+b of the 32-byte K slice holds bit
// m+8b.  That is a fixed permutation of k inside each 32-wide slice, applied identically to both
// operands, so the sum over k is unchanged and the expansion costs one shift and one AND per
// four bytes.  Every match contributes 128*128 = 2^14; the int32 accumulator holds count * 2^14
// exactly for counts < 2^17 (N <= 131072; checked by the launcher), and count = acc >> 14.
//
// CTA = one SM (512 TMEM columns), persistent over 128 x 256 tiles (rows i x rows j), 18 warps:
//   warps 0-3   epilogue: tcgen05.ld the accumulator rows, test the relation bit U[i][j], update the
//               shared-memory histogram (global atomics for rare large intervals)
//   warp  4     TMEM allocation + the single MMA-issuing thread
//   warp  5     loader: one thread issues the TMA tensor copies (cp.async.bulk.tensor, 64B swizzle)
//               that stage the bit rows, GK k-steps (64 bytes per row) at a time
//   warps 6-17  expanders: 384 threads, one operand row each (128 rows of U, 256 rows of L)
// Pipelines: NB bit-row buffers (bfull/bempty), NS shared-memory operand stages (full/empty; the
// MMA warp releases a stage with tcgen05.commit), two TMEM accumulator buffers (tfull/tempty).
#include <cuda.h>

#include "cs_common.cuh"

namespace cs {

namespace {

constexpr int TM = 128;                 // tile rows i (MMA M)
constexpr int TN = 256;                 // tile rows j (MMA N)
constexpr int KSTEP = 128;              // k per stage = 128 bytes of int8 = 4 MMAs of K = 32
constexpr int NS = 3;                   // shared-memory stages of expanded operands
constexpr int GK = 4;                   // k-steps per staged group of bit rows (64 bytes per row)
constexpr int BROW = GK * 16;           // bytes per staged bit row (TMA box inner extent, 64B swizzle)
constexpr int NB = 3;                   // bit-row buffers
constexpr int BITS_BYTES = (TM + TN) * BROW;
constexpr int A_BYTES = TM * KSTEP;     // 16 KiB
constexpr int B_BYTES = TN * KSTEP;     // 32 KiB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int HS = 2048;                // shared-memory histogram bins
constexpr int EPI_WARPS = 4, MMA_WARP = 4, LOAD_WARP = 5, EXP_WARP0 = 6, EXP_WARPS = 12;
constexpr int THREADS = (EPI_WARPS + 2 + EXP_WARPS) * 32;   // 576
constexpr int EXP_THREADS = EXP_WARPS * 32;                 // 384 = TM + TN
constexpr int SMEM_BYTES = NS * STAGE_BYTES + NB * BITS_BYTES + HS * 4 + 256;
constexpr int SCALE_SHIFT = 14;         // every match adds 128 * 128

static_assert(EXP_THREADS == TM + TN, "one expander thread per operand row");
// a thread may run at most NS k-steps ahead of the slowest warp; keeping that below one group keeps
// every thread within one phase of the bit-buffer barriers
static_assert(NS <= GK, "stage ring must not outrun a bit-row group");

// instruction descriptor, kind::i8: D = S32 (2 at bit 4), A = B = U8 (0), both K-major,
// N >> 3 at bit 17, M >> 4 at bit 24
constexpr uint32_t IDESC = (2u << 4) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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

__device__ __forceinline__ void mma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum)
        : "memory");
}
__device__ __forceinline__ void mma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
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
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

struct Tile {
    int I, J;   // 128-row block of i, 256-row block of j
};
// tiles of one causet ordered by decreasing number of k-steps (2J + 2 - I); nTJ(nTJ+1) tiles
__device__ __forceinline__ Tile tile_from_index(int64_t t, int nTJ)
{
    int64_t q = (int64_t)((sqrt(4.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((q + 1) * (q + 2) <= t) q++;
    while (q * (q + 1) > t) q--;
    const int r = (int)(t - q * (q + 1));
    const int p = nTJ - 1 - (int)q;
    if (r < (int)q + 1) return Tile{2 * r, p + r};                 // d = 2p+1
    const int idx = r - ((int)q + 1);
    return Tile{2 * idx + 1, p + idx};                             // d = 2p
}

__global__ void __launch_bounds__(THREADS, 1)
k_interval_tensor(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapL,
                  const uint64_t *__restrict__ bits,
                  int64_t B, int64_t N, int64_t stride, int64_t kmax,
                  int64_t row_begin, int64_t row_end,
                  unsigned long long *__restrict__ hist, unsigned long long *__restrict__ nrel)
{
    extern __shared__ __align__(1024) unsigned char smem[];   // typed shared base: STS/ATOMS, not generic
    unsigned char *s_stage = smem;
    unsigned char *s_bits = smem + NS * STAGE_BYTES;
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(smem + NS * STAGE_BYTES + NB * BITS_BYTES);
    uint64_t *s_full = reinterpret_cast<uint64_t *>(smem + NS * STAGE_BYTES + NB * BITS_BYTES + HS * 4);
    uint64_t *s_empty = s_full + NS;
    uint64_t *s_tfull = s_empty + NS;     // [2]
    uint64_t *s_tempty = s_tfull + 2;     // [2]
    uint64_t *s_bfull = s_tempty + 2;     // [NB] staged bit rows have landed
    uint64_t *s_bempty = s_bfull + NB;    // [NB] every expander warp is done with the buffer
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(s_bempty + NB);
    unsigned long long *s_nrel = reinterpret_cast<unsigned long long *>(s_tmem + 2);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nTJ = (int)((N + TN - 1) / TN);
    const int64_t tiles_per = (int64_t)nTJ * (nTJ + 1);
    const int64_t total_tiles = tiles_per * B;
    const int hs = (int)((kmax + 1 < HS) ? (kmax + 1) : HS);
    const int64_t hist_len = kmax + 1;

    if (tid == 0) {
        for (int s = 0; s < NS; s++) {
            mbar_init(&s_full[s], EXP_WARPS);
            mbar_init(&s_empty[s], 1);
        }
        for (int b = 0; b < NB; b++) {
            mbar_init(&s_bfull[b], 1);
            mbar_init(&s_bempty[b], EXP_WARPS);
        }
        for (int a = 0; a < 2; a++) {
            mbar_init(&s_tfull[a], 1);
            mbar_init(&s_tempty[a], EPI_WARPS * 32);
        }
        *s_nrel = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int b = tid; b < HS; b += THREADS) s_hist[b] = 0;
    if (warp == MMA_WARP) {   // allocate all 512 TMEM columns (one CTA per SM by shared-memory size)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(s_tmem)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *s_tmem;

    // every role walks the same static schedule: tile t = blockIdx.x, + gridDim.x, ...
    if (warp >= EXP_WARP0) {
        // ===================================== expanders =====================================
        const int e = tid - EXP_WARP0 * 32;
        const bool isA = e < TM;
        const int r = isA ? e : e - TM;
        const uint32_t rows = isA ? TM : TN;
        uint32_t it = 0;   // global k-step counter (stage ring position)
        uint32_t grp = 0;  // global group counter (bit-buffer ring position)
        // TMA 64B swizzle: 16-byte chunk c of row e sits at chunk c ^ ((e >> 1) & 3)
        const unsigned char *my_bits = s_bits + (isA ? 0 : TM * BROW) + r * BROW;
        const int swz = (r >> 1) & 3;
        for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
            const int64_t bidx = t / tiles_per;
            const Tile tc = tile_from_index(t - bidx * tiles_per, nTJ);
            if ((int64_t)tc.I * TM >= row_end || (int64_t)(tc.I + 1) * TM <= row_begin) continue;
            const int ks0 = tc.I, ks1 = 2 * tc.J + 1;            // inclusive k-step range
            const int ngroups = (ks1 - ks0 + GK) / GK;
            for (int g = 0; g < ngroups; g++, grp++) {
                const int b = grp % NB;
                mbar_wait(&s_bfull[b], (grp / NB) & 1);
                const int kcount = (ks1 - (ks0 + g * GK) + 1 < GK) ? (ks1 - (ks0 + g * GK) + 1) : GK;
                for (int c = 0; c < kcount; c++, it++) {
                    const uint4 cur = *reinterpret_cast<const uint4 *>(my_bits + b * BITS_BYTES + ((c ^ swz) << 4));
                    const int s = it % NS;
                    mbar_wait(&s_empty[s], ((it / NS) & 1) ^ 1);
                    unsigned char *dst = s_stage + s * STAGE_BYTES + (isA ? 0 : A_BYTES) + r * 16;
                    const uint32_t xs[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        const uint32_t x = xs[q];
                        uint4 lo, hi;
                        lo.x = (x << 7) & 0x80808080u;
                        lo.y = (x << 6) & 0x80808080u;
                        lo.z = (x << 5) & 0x80808080u;
                        lo.w = (x << 4) & 0x80808080u;
                        hi.x = (x << 3) & 0x80808080u;
                        hi.y = (x << 2) & 0x80808080u;
                        hi.z = (x << 1) & 0x80808080u;
                        hi.w = x & 0x80808080u;
                        *reinterpret_cast<uint4 *>(dst + (2 * q) * rows * 16) = lo;
                        *reinterpret_cast<uint4 *>(dst + (2 * q + 1) * rows * 16) = hi;
                    }
                    fence_proxy_async();          // generic-proxy stores -> visible to the tensor core
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(&s_full[s]);                          // one arrival per warp
                        // last chunk of the buffer has been loaded AND consumed by every lane (the
                        // stores above depend on it): hand the bit buffer back to the loader
                        if (c == kcount - 1) mbar_arrive(&s_bempty[b]);
                    }
                }
            }
        }
    } else if (warp == LOAD_WARP) {
        // ===================================== TMA loader ====================================
        if (lane == 0) {
            uint32_t grp = 0;
            for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
                const int64_t bidx = t / tiles_per;
                const Tile tc = tile_from_index(t - bidx * tiles_per, nTJ);
                if ((int64_t)tc.I * TM >= row_end || (int64_t)(tc.I + 1) * TM <= row_begin) continue;
                const int ks0 = tc.I, ks1 = 2 * tc.J + 1;
                const int ngroups = (ks1 - ks0 + GK) / GK;
                for (int g = 0; g < ngroups; g++, grp++) {
                    const int b = grp % NB;
                    mbar_wait(&s_bempty[b], ((grp / NB) & 1) ^ 1);
                    mbar_arrive_expect_tx(&s_bfull[b], (uint32_t)BITS_BYTES);   // out-of-bounds is zero-filled
                    unsigned char *dst = s_bits + b * BITS_BYTES;
                    const int c0 = (ks0 + g * GK) * 16;
                    tma_load_3d(dst, &mapU, c0, tc.I * TM, (int)bidx, &s_bfull[b]);
                    tma_load_3d(dst + TM * BROW, &mapL, c0, tc.J * TN, (int)bidx, &s_bfull[b]);
                }
            }
        }
    } else if (warp == MMA_WARP) {
        // ===================================== MMA issuer ====================================
        if (lane == 0) {
            uint32_t it = 0, tile_seq = 0;
            for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
                const int64_t bidx = t / tiles_per;
                const Tile tc = tile_from_index(t - bidx * tiles_per, nTJ);
                if ((int64_t)tc.I * TM >= row_end || (int64_t)(tc.I + 1) * TM <= row_begin) continue;
                const int ks0 = tc.I, ks1 = 2 * tc.J + 1;
                const uint32_t a = tile_seq & 1;
                mbar_wait(&s_tempty[a], ((tile_seq >> 1) & 1) ^ 1);      // epilogue has drained buffer a
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + a * TN;
                for (int ks = ks0; ks <= ks1; ks++, it++) {
                    const int s = it % NS;
                    mbar_wait(&s_full[s], (it / NS) & 1);
                    tc_fence_after();
                    const uint32_t a_addr = smem_u32(s_stage + s * STAGE_BYTES);
                    const uint32_t b_addr = a_addr + A_BYTES;
#pragma unroll
                    for (int q = 0; q < KSTEP / 32; q++) {
                        const uint64_t ad = make_desc(a_addr + q * 2 * TM * 16, TM * 16, 128);
                        const uint64_t bd = make_desc(b_addr + q * 2 * TN * 16, TN * 16, 128);
                        mma_i8(d_tmem, ad, bd, IDESC, (ks > ks0 || q > 0) ? 1u : 0u);
                    }
                    mma_commit(&s_empty[s]);                              // stage s free once these MMAs retire
                }
                mma_commit(&s_tfull[a]);                                  // accumulator complete
                tile_seq++;
            }
        }
    } else {
        // ===================================== epilogue ======================================
        uint32_t tile_seq = 0;
        unsigned long long my_nrel = 0;
        const uint32_t hist_saddr = smem_u32(s_hist);
        const uint32_t kmax32 = (uint32_t)kmax;
        int64_t cur_batch = -1;
        for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
            const int64_t bidx = t / tiles_per;
            const Tile tc = tile_from_index(t - bidx * tiles_per, nTJ);
            if ((int64_t)tc.I * TM >= row_end || (int64_t)(tc.I + 1) * TM <= row_begin) continue;
            if (bidx != cur_batch) {   // per-causet histograms: flush before switching
                if (cur_batch >= 0 && B > 1) {
                    asm volatile("bar.sync 1, 128;");
                    for (int b = tid; b < hs; b += EPI_WARPS * 32) {
                        uint32_t v = s_hist[b];
                        if (v) { atomicAdd(&hist[cur_batch * hist_len + b], (unsigned long long)v); s_hist[b] = 0; }
                    }
                    asm volatile("bar.sync 1, 128;");
                }
                cur_batch = bidx;
            }
            const int64_t i = (int64_t)tc.I * TM + tid;          // this thread's row = TMEM lane
            const bool row_ok = i < N && i >= row_begin && i < row_end;
            uint64_t rel[4] = {0, 0, 0, 0};
            if (row_ok) {
                const uint64_t *urow = bits + bidx * N * stride + i * stride;
#pragma unroll
                for (int w = 0; w < 4; w++) {
                    const int64_t wi = (int64_t)tc.J * 4 + w;
                    if (wi < stride) rel[w] = __ldg(urow + wi);
                }
            }
            unsigned long long *ghist = hist + cur_batch * hist_len;
            const uint32_t a = tile_seq & 1;
            mbar_wait(&s_tfull[a], (tile_seq >> 1) & 1);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(warp * 32) << 16) + a * TN;
#pragma unroll
            for (int c8 = 0; c8 < TN / 32; c8++) {
                const uint32_t rel32 = (uint32_t)(rel[c8 >> 1] >> (32 * (c8 & 1)));
                if (!__any_sync(0xffffffffu, rel32 != 0)) continue;
                uint32_t v[32];
                tmem_ld32(taddr + c8 * 32, v);
                if (rel32 == 0) continue;
                my_nrel += __popc(rel32);
                // branch-free: two predicated reductions per element (a divergent if/else here costs
                // one serialized pass per column in which any lane has a related pair)
#pragma unroll
                for (int c = 0; c < 32; c++) {
                    const uint32_t cnt = v[c] >> SCALE_SHIFT;
                    const uint32_t on = (rel32 >> c) & 1u;
                    const uint32_t small = on & (cnt < (uint32_t)hs ? 1u : 0u);
                    const uint32_t big = on & (small ^ 1u) & (cnt <= kmax32 ? 1u : 0u);
                    asm volatile(
                        "{\n"
                        ".reg .pred ps, pb;\n"
                        "setp.ne.u32 ps, %0, 0;\n"
                        "setp.ne.u32 pb, %1, 0;\n"
                        "@ps red.shared.add.u32 [%2], 1;\n"
                        "@pb red.global.add.u64 [%3], 1;\n"
                        "}\n" ::"r"(small),
                        "r"(big), "r"(hist_saddr + cnt * 4u), "l"(ghist + cnt)
                        : "memory");
                }
            }
            tc_fence_before();
            mbar_arrive(&s_tempty[a]);
            tile_seq++;
        }
        // final flush by the epilogue warps
        asm volatile("bar.sync 1, 128;");
        if (cur_batch >= 0) {
            for (int b = tid; b < hs; b += EPI_WARPS * 32) {
                uint32_t v = s_hist[b];
                if (v) atomicAdd(&hist[cur_batch * hist_len + b], (unsigned long long)v);
            }
        }
        if (nrel && B == 1) {
#pragma unroll
            for (int s = 16; s >= 1; s >>= 1) my_nrel += __shfl_xor_sync(0xffffffffu, my_nrel, s);
            if (lane == 0 && my_nrel) atomicAdd(nrel, my_nrel);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == MMA_WARP) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base));
    }
}

}  // namespace

bool interval_tensor_available() { return true; }
size_t interval_tensor_scratch_bytes(int64_t, int64_t) { return 0; }

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
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

// bit matrix [B][N][stride uint64] seen as bytes: dims {stride*8, N, B}; box {64 bytes, rows, 1}
static int make_bits_map(CUtensorMap *map, const uint64_t *base, int64_t B, int64_t N, int64_t stride, int rows)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled entry point not available");
        return CS_ERR_CUDA;
    }
    cuuint64_t gdim[3] = {(cuuint64_t)(stride * 8), (cuuint64_t)N, (cuuint64_t)B};
    cuuint64_t gstr[2] = {(cuuint64_t)(stride * 8), (cuuint64_t)(N * stride * 8)};
    cuuint32_t box[3] = {(cuuint32_t)BROW, (cuuint32_t)rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<uint64_t *>(base), gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed (%d)", (int)r);
        return CS_ERR_CUDA;
    }
    return CS_OK;
}

int launch_interval_tensor(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                           int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                           void *, size_t, cudaStream_t st)
{
    if (N > ((int64_t)1 << 17)) return CS_ERR_ARG;   // count * 2^14 must stay below 2^31
    static PerDeviceFlag attr_set;
    const int dev = current_device();
    if (!attr_set.get(dev)) {
        CS_CUDA(cudaFuncSetAttribute(k_interval_tensor, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
        attr_set.set(dev);
    }
    const int64_t stride = row_stride_words(N);
    CUtensorMap mapU, mapL;
    int rc = make_bits_map(&mapU, bits, B, N, stride, TM);
    if (rc) return rc;
    rc = make_bits_map(&mapL, bitsT, B, N, stride, TN);
    if (rc) return rc;
    const int64_t nTJ = (N + TN - 1) / TN;
    const int64_t total = nTJ * (nTJ + 1) * B;
    int64_t grid = sm_count();
    if (grid > total) grid = total;
    if (grid < 1) grid = 1;
    k_interval_tensor<<<(unsigned)grid, THREADS, SMEM_BYTES, st>>>(
        mapU, mapL, bits, B, N, stride, kmax, row_begin, row_end,
        reinterpret_cast<unsigned long long *>(hist), reinterpret_cast<unsigned long long *>(nrel));
    CS_LAUNCHED("k_interval_tensor");
    return CS_OK;
}

}  // namespace cs
