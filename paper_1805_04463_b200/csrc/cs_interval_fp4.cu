// cs_interval_fp4.cu -- stage a2, tensor route with 4-bit operands (tcgen05.mma kind::mxf4).
//
// Same contraction and the same CTA skeleton as cs_interval_tensor.cu (int8): count(i,j) =
// sum_k U[i][k] * L[j][k] over the K blocks between the I block and the J block (Fig. 4.2 caption
// PAPER.md:1768; Alg. 20 line 9).  The int8 kernel is bound by shared-memory
// bandwidth (operand bytes written by the expanders + read by the MMA); here a bit becomes the
// E2M1 nibble 0b0010 (= 1.0) instead of a byte, which halves the operand bytes per k and doubles
// the MMA rate: a 48 KB stage now covers 256 k.  With x a 32-bit slice of a row, output word
// m = ((x << 1) >> m) & 0x22222222 (m = 0..3): nibble n of word m holds bit 4n+m -- again a fixed
// permutation of k inside the slice, applied to both operands.  Block scales are UE8M0 = 2^0
// (byte 0x7F) everywhere, written once into TMEM.  Products are 0 or 1 and the fp32 accumulator
// is exact for counts < 2^24 (measured: identical histograms to the int8 and POPC routes).
//
// TMEM: one 256-column fp32 accumulator + 2 x 32 columns of scale factors (a second accumulator
// does not fit next to them), so the epilogue is not overlapped with the next tile's MMAs; it is
// branch-free and short (8 tcgen05.ld + 512 predicated reductions per thread).
#include <cuda.h>

#include "cs_common.cuh"

namespace cs {

namespace {

constexpr int TM = 128;                 // tile rows i (MMA M)
constexpr int TN = 256;                 // tile rows j (MMA N)
constexpr int KSTEP = 256;              // k per stage = 128 bytes of E2M1 = 4 MMAs of K = 64
constexpr int KBYTES = KSTEP / 2;       // operand bytes per row per stage
constexpr int NS = 4;                   // stages: B operand in shared memory, A operand in TMEM
constexpr int GK = 2;                   // stages per staged group of bit rows (64 bytes per row)
constexpr int BROW = GK * 32;           // bytes per staged bit row (TMA box inner extent, 64B swizzle)
constexpr int NB = 2;                   // bit-row buffers
constexpr int EPITCH = 20;              // words per thread row of the epilogue staging area (16 counts + pad)
constexpr int EPI_BYTES = 256 * EPITCH * 4;
constexpr int BITS_BYTES = (TM + TN) * BROW;
constexpr int B_BYTES = TN * KBYTES;    // 32 KiB
constexpr int STAGE_BYTES = B_BYTES;     // the A operand of a stage lives in 32 TMEM columns
constexpr int HS = 2048;                // shared-memory histogram bins
constexpr int EPI_WARPS = 8, MMA_WARP = 8, LOAD_WARP = 9, EXP_WARP0 = 10, EXP_WARPS = 12;
constexpr int THREADS = (EPI_WARPS + 2 + EXP_WARPS) * 32;   // 576
constexpr int EXP_THREADS = EXP_WARPS * 32;                 // 384 = TM + TN
constexpr int SMEM_BYTES = NS * STAGE_BYTES + NB * BITS_BYTES + EPI_BYTES + HS * 4 + 256;

static_assert(EXP_THREADS == TM + TN, "one expander thread per operand row");


// block-scaled instruction descriptor, kind::mxf4: A = B = E2M1 (1 at bits 7 and 10), both K-major,
// N >> 3 at bit 17, scale format UE8M0 (1 at bit 23), M >> 4 at bit 24, scale-factor ids 0, K = 64
constexpr uint32_t IDESC = (1u << 7) | (1u << 10) | ((uint32_t)(TN >> 3) << 17) | (1u << 23) | ((uint32_t)(TM >> 4) << 24);
constexpr uint32_t SFA_COL = 256, SFB_COL = 288;   // TMEM columns of the (constant) scale factors
constexpr uint32_t A_COL = 320;                    // TMEM ring of the A operand: NS x 32 columns
static_assert(A_COL + NS * 32 <= 512, "TMEM columns");

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

__device__ __forceinline__ void mma_mxf4(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accum,
                                         uint32_t sfa, uint32_t sfb)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%5], [%6], p;\n"
        "}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accum), "r"(sfa), "r"(sfb)
        : "memory");
}
__device__ __forceinline__ void tmem_st32_const(uint32_t taddr, uint32_t val)
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, "
        "%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};\n" ::"r"(taddr),
        "r"(val)
        : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void mma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};\n" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]),
        "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]),
        "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31])
        : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
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
k_interval_fp4(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapL,
                  const uint64_t *__restrict__ bits,
                  int64_t B, int64_t N, int64_t stride, int64_t kmax,
                  int64_t row_begin, int64_t row_end,
                  unsigned long long *__restrict__ hist, unsigned long long *__restrict__ nrel)
{
    extern __shared__ __align__(1024) unsigned char smem[];   // typed shared base: STS/ATOMS, not generic
    unsigned char *s_stage = smem;
    unsigned char *s_bits = smem + NS * STAGE_BYTES;
    uint32_t *s_epi = reinterpret_cast<uint32_t *>(smem + NS * STAGE_BYTES + NB * BITS_BYTES);
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(smem + NS * STAGE_BYTES + NB * BITS_BYTES + EPI_BYTES);
    uint64_t *s_full = reinterpret_cast<uint64_t *>(smem + NS * STAGE_BYTES + NB * BITS_BYTES + EPI_BYTES + HS * 4);
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
    if (warp < 4) {   // constant block scales UE8M0 = 2^0 in every byte of the scale-factor columns
        const uint32_t sf = tmem_base + ((uint32_t)(warp * 32) << 16) + SFA_COL;
        tmem_st32_const(sf, 0x7F7F7F7Fu);
        tmem_st32_const(sf + 32, 0x7F7F7F7Fu);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    // every role walks the same static schedule: tile t = blockIdx.x, + gridDim.x, ...
    if (warp >= EXP_WARP0) {
        // ===================================== expanders =====================================
        // expander warps 0-3 own the A rows (row = TMEM lane: warp w may only touch lanes 32 (w % 4) ..),
        // warps 4-11 the B rows
        const int ew = warp - EXP_WARP0;
        const bool isA = ew < 4;
        const int r = isA ? ((warp & 3) * 32 + lane) : ((ew - 4) * 32 + lane);
        uint32_t it = 0;   // global k-step counter (stage ring position)
        uint32_t grp = 0;  // global group counter (bit-buffer ring position)
        // TMA 64B swizzle: 16-byte chunk c of row e sits at chunk c ^ ((e >> 1) & 3)
        const unsigned char *my_bits = s_bits + (isA ? 0 : TM * BROW) + r * BROW;
        const int swz = (r >> 1) & 3;
        for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
            const int64_t bidx = t / tiles_per;
            const Tile tc = tile_from_index(t - bidx * tiles_per, nTJ);
            if ((int64_t)tc.I * TM >= row_end || (int64_t)(tc.I + 1) * TM <= row_begin) continue;
            const int ks0 = tc.I >> 1, ks1 = tc.J;                // inclusive range of 256-k stages
            const int ngroups = (ks1 - ks0 + GK) / GK;
            for (int g = 0; g < ngroups; g++, grp++) {
                const int b = grp % NB;
                mbar_wait(&s_bfull[b], (grp / NB) & 1);
                const int kcount = (ks1 - (ks0 + g * GK) + 1 < GK) ? (ks1 - (ks0 + g * GK) + 1) : GK;
                for (int c = 0; c < kcount; c++, it++) {
                    const uint4 cur0 = *reinterpret_cast<const uint4 *>(my_bits + b * BITS_BYTES + (((2 * c) ^ swz) << 4));
                    const uint4 cur1 = *reinterpret_cast<const uint4 *>(my_bits + b * BITS_BYTES + (((2 * c + 1) ^ swz) << 4));
                    const int s = it % NS;
                    mbar_wait(&s_empty[s], ((it / NS) & 1) ^ 1);
                    const uint32_t xs[8] = {cur0.x, cur0.y, cur0.z, cur0.w, cur1.x, cur1.y, cur1.z, cur1.w};
                    if (isA) {
                        // 32 k -> 4 words of E2M1 nibbles (1.0 = 0b0010); 8 slices -> the 32 TMEM columns of stage s
                        uint32_t w[32];
#pragma unroll
                        for (int q = 0; q < 8; q++) {
                            const uint32_t x = xs[q];
                            w[4 * q + 0] = (x << 1) & 0x22222222u;
                            w[4 * q + 1] = x & 0x22222222u;
                            w[4 * q + 2] = (x >> 1) & 0x22222222u;
                            w[4 * q + 3] = (x >> 2) & 0x22222222u;
                        }
                        tmem_st32(tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + A_COL + s * 32, w);
                        tc_fence_before();
                    } else {
                        unsigned char *dst = s_stage + s * STAGE_BYTES + r * 16;
#pragma unroll
                        for (int q = 0; q < 8; q++) {     // 32 k -> one 16-byte chunk of E2M1 nibbles
                            const uint32_t x = xs[q];
                            uint4 w;
                            w.x = (x << 1) & 0x22222222u;
                            w.y = x & 0x22222222u;
                            w.z = (x >> 1) & 0x22222222u;
                            w.w = (x >> 2) & 0x22222222u;
                            *reinterpret_cast<uint4 *>(dst + q * TN * 16) = w;
                        }
                        fence_proxy_async();          // generic-proxy stores -> visible to the tensor core
                    }
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
                const int ks0 = tc.I >> 1, ks1 = tc.J;
                const int ngroups = (ks1 - ks0 + GK) / GK;
                for (int g = 0; g < ngroups; g++, grp++) {
                    const int b = grp % NB;
                    mbar_wait(&s_bempty[b], ((grp / NB) & 1) ^ 1);
                    mbar_arrive_expect_tx(&s_bfull[b], (uint32_t)BITS_BYTES);   // out-of-bounds is zero-filled
                    unsigned char *dst = s_bits + b * BITS_BYTES;
                    const int c0 = (ks0 + g * GK) * 32;
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
                const int ks0 = tc.I >> 1, ks1 = tc.J;
                mbar_wait(&s_tempty[0], (tile_seq & 1) ^ 1);             // epilogue has drained the accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base;
                for (int ks = ks0; ks <= ks1; ks++, it++) {
                    const int s = it % NS;
                    mbar_wait(&s_full[s], (it / NS) & 1);
                    tc_fence_after();
                    const uint32_t b_addr = smem_u32(s_stage + s * STAGE_BYTES);
#pragma unroll
                    for (int q = 0; q < KBYTES / 32; q++) {       // K = 64 per MMA: 8 TMEM columns of A, 2 chunks of B
                        const uint64_t bd = make_desc(b_addr + q * 2 * TN * 16, TN * 16, 128);
                        mma_mxf4(d_tmem, tmem_base + A_COL + s * 32 + q * 8, bd, IDESC, (ks > ks0 || q > 0) ? 1u : 0u,
                                 tmem_base + SFA_COL, tmem_base + SFB_COL);
                    }
                    mma_commit(&s_empty[s]);                              // stage s free once these MMAs retire
                }
                mma_commit(&s_tfull[0]);                                  // accumulator complete
                tile_seq++;
            }
        }
    } else {
        // ===================================== epilogue ======================================
        uint32_t tile_seq = 0;
        unsigned long long my_nrel = 0;
        const uint32_t kmax32 = (uint32_t)kmax;
        int64_t cur_batch = -1;
        for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
            const int64_t bidx = t / tiles_per;
            const Tile tc = tile_from_index(t - bidx * tiles_per, nTJ);
            if ((int64_t)tc.I * TM >= row_end || (int64_t)(tc.I + 1) * TM <= row_begin) continue;
            if (bidx != cur_batch) {   // per-causet histograms: flush before switching
                if (cur_batch >= 0 && B > 1) {
                    asm volatile("bar.sync 1, 256;");
                    for (int b = tid; b < hs; b += EPI_WARPS * 32) {
                        uint32_t v = s_hist[b];
                        if (v) { atomicAdd(&hist[cur_batch * hist_len + b], (unsigned long long)v); s_hist[b] = 0; }
                    }
                    asm volatile("bar.sync 1, 256;");
                }
                cur_batch = bidx;
            }
            const int quarter = warp & 3, colhalf = warp >> 2;   // TMEM lane quarter; which 128 columns
            const int64_t i = (int64_t)tc.I * TM + quarter * 32 + lane;   // this thread's row = TMEM lane
            const bool row_ok = i < N && i >= row_begin && i < row_end;
            uint64_t rel[2] = {0, 0};                            // relation bits of this warp's 128 columns
            if (row_ok) {
                const uint64_t *urow = bits + bidx * N * stride + i * stride;
#pragma unroll
                for (int w = 0; w < 2; w++) {
                    const int64_t wi = (int64_t)tc.J * 4 + colhalf * 2 + w;
                    if (wi < stride) rel[w] = __ldg(urow + wi);
                }
            }
            unsigned long long *ghist = hist + cur_batch * hist_len;
            mbar_wait(&s_tfull[0], tile_seq & 1);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + colhalf * 128;
            uint32_t *my = s_epi + tid * EPITCH;
            auto tally = [&](uint32_t word) {
                const uint32_t cnt = (uint32_t)__uint_as_float(word);   // products are 0 or 1: exact in fp32
                if (cnt < (uint32_t)hs) atomicAdd(&s_hist[cnt], 1u);
                else if (cnt <= kmax32) atomicAdd(&ghist[cnt], 1ULL);
            };
#pragma unroll
            for (int c16 = 0; c16 < 8; c16++) {
                const uint32_t rel16 = (uint32_t)(rel[c16 >> 2] >> (16 * (c16 & 3))) & 0xFFFFu;
                if (!__any_sync(0xffffffffu, rel16 != 0)) continue;
                uint32_t v[16];
                tmem_ld16(taddr + c16 * 16, v);
                if (rel16 == 0) continue;
                my_nrel += __popc(rel16);
                // Stage the 16 counts in this thread's private shared-memory row, then visit only the
                // columns whose relation bit is set, two per iteration (work ~ related pairs, not
                // columns; a predicated reduction per column compiles to a divergent branch per column).
#pragma unroll
                for (int c4 = 0; c4 < 4; c4++)
                    *reinterpret_cast<uint4 *>(my + 4 * c4) = make_uint4(v[4 * c4], v[4 * c4 + 1], v[4 * c4 + 2], v[4 * c4 + 3]);
                uint32_t m = rel16;
                while (m) {
                    const int c0 = __ffs(m) - 1;
                    m &= m - 1;
                    const bool two = m != 0;
                    const int c1 = two ? __ffs(m) - 1 : c0;
                    m &= m - 1;
                    const uint32_t w0 = my[c0], w1 = my[c1];
                    tally(w0);
                    if (two) tally(w1);
                }
            }
            tc_fence_before();
            mbar_arrive(&s_tempty[0]);
            tile_seq++;
        }
        // final flush by the epilogue warps
        asm volatile("bar.sync 1, 256;");
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

int launch_interval_fp4(const uint64_t *bits, const uint64_t *bitsT, int64_t B, int64_t N, int64_t kmax,
                           int64_t row_begin, int64_t row_end, int64_t *hist, int64_t *nrel,
                           void *, size_t, cudaStream_t st)
{
    if (N > ((int64_t)1 << 24)) return CS_ERR_ARG;   // counts must stay exact in fp32
    static PerDeviceFlag attr_set;
    const int dev = current_device();
    if (!attr_set.get(dev)) {
        CS_CUDA(cudaFuncSetAttribute(k_interval_fp4, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
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
    k_interval_fp4<<<(unsigned)grid, THREADS, SMEM_BYTES, st>>>(
        mapU, mapL, bits, B, N, stride, kmax, row_begin, row_end,
        reinterpret_cast<unsigned long long *>(hist), reinterpret_cast<unsigned long long *>(nrel));
    CS_LAUNCHED("k_interval_fp4");
    return CS_OK;
}

}  // namespace cs
