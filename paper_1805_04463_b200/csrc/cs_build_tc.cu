// cs_build_tc.cu -- stage a1 on the tensor cores: every predicate of the library as the sign of a bilinear form
// (flat cone in 1+1 .. 4+1 dimensions, FLRW Eq. 7.7, 3+1 de Sitter as in cs_predicates.cuh; the 1+1 light cone and the
// 1+1 de Sitter slab in derived coordinates, TcFast below).
//
// The sign of the interval between i and j is the sign of
//     T(i, j) = h_i + h_j + sum_c P_c(i) F_c(j)          (cs_predicates.cuh, Fast<GEOM, DIM>)
// i.e. one entry of a rank-(NP + 2) matrix product.  Every fp32 input v is split exactly into three bf16 pieces
// v = hi + mid + lo (round to nearest each time: |mid| <= 2^-8 |v|, |lo| <= 2^-16 |v|); a product P F is then the sum
// of nine piece products, each exact in fp32, of which the six not smaller than 2^-16 |P F| are kept:
//     hi hi | hi mid, mid hi | mid mid, hi lo, lo hi          (dropped: mid lo, lo mid, lo lo <= 2.01 * 2^-24 |P F|)
// and h_i + h_j enters as (h pieces of i) x 1 + 1 x (h pieces of j).  That is K = 6 NP + 6 <= 32 (48 for five or six
// products) bf16 columns per point, and T for a 128 x 256 block of pairs is two (three) tcgen05.mma kind::f16
// instructions with fp32 accumulation in TMEM -- 1/32 of what the FMA pipes need for the same block.
//
// What the tensor core returns is a value `a` with |a - T| <= E = E_in + E_acc (u = 2^-24, C = largest |component| of
// the tile):
//   E_in   the inputs of the fp32 prefilter (the same fp64 -> fp32 conversions as in cs_build.cu; Fast::MARGIN / 2 u C^2
//          covers them with room) and the dropped piece products (<= 2.01 NP u C^2): (MARGIN / 2 + 3 NP) u C^2.
//   E_acc  the accumulation inside the tensor core, whose width and order are not documented.  Model taken (the one
//          published analyses of earlier generations found, and what the probe below measures here): an instruction
//          aligns its 16 products and the accumulator to the largest exponent among them, keeps at least 24 bits, adds
//          exactly and rounds once -- every addend loses less than 2^-23 of the largest one.  For a pair near the cone
//          (|T| small, the only pairs whose sign an error can change) the largest addend is at most
//          M = max(|h_i|, |h_j|, |P_c(i) F_c(j)|), bounded per tile from per-128-point maxima, so
//          E_acc <= (K + 2) 2 u M over the K / 16 instructions; for a pair with |T| >= M the same model gives a relative
//          error of (K + 2) 2 u, which cannot change a sign either.
// The margin is m = (4 (K + 2) M + (MARGIN / 2 + 3 NP) C^2) u, i.e. TWICE the modelled accumulation loss.
// `cs_a1_tensor_probe` measures on real tiles |a - T| against the fp64 value, |a - S| against the exact sum S of the
// operand products, and the largest |a - T| / m (profiles/r2b_a1_tensor.md: the accumulation alone loses up to 14 u C^2
// -- the tensor core does truncate --, |a - T| / m stays below 0.08).
//     |a| > m   =>   sign(a) = sign(T), and |T| is far outside the rounding of the fp64 expression of the header
//                    (2^-46 C^2): related iff a > 0
//     anything else (NaN included): the 32 pairs of that ROW of the block are re-evaluated with the fp64 expression.
// As in cs_build.cu a tile takes the prefilter only if dt >= 0 is known for every pair it keeps (time order per
// tile, checked on the doubles by the prep kernel), 2^-40 <= C <= 2^40 and every point is finite and passes
// Fast::convert; otherwise m = +inf and every row goes to fp64.  The output is bit-identical to the fp64 evaluation
// as long as the model above holds; the parity tests compare every bit with the oracle.
//
// Kernels: k_tc_prep (one thread per point: conversion, pieces, both operand rows in the UMMA canonical K-major
// layout, a padded copy of the coordinates, per-128-point summaries), k_tc_tiles (one thread per tile: its (I, J), causet
// and margin) and k_causal_tc (persistent, one CTA per SM):
//   loader (1 thread)    bulk copies of the tile's operand rows and coordinates into a 3-deep ring
//   MMA issuer (1 thread) K / 16 tcgen05.mma (M = 128, N = 256) per half tile into two TMEM accumulators
//   16 epilogue warps    each 32 rows x 64 columns of a half: tcgen05.ld (lane = row), the 32 sign bits of the row into
//                        one word (funnel shift on the ALU pipe; TC_NF of them through fma.sat on the idle FMA pipe),
//                        min |a| (one FMNMX3 per two pairs), fp64 rows if the minimum is inside the band, the shuffle
//                        butterfly for the transposed output (interleaved with the next block's extraction), both
//                        words staged in shared memory
//   2 writer warps       the staged 256 x 256 tile to global memory as 32-byte row segments; the mirrored tile of an
//                        off-diagonal tile as two TMA tile stores from a constant zero tile.
// The kernel is bound by instruction issue / the ALU pipe: 1.5 instructions per pair are the floor of this scheme.
#include <cuda.h>
#include <cuda_bf16.h>

#include <type_traits>

#include "cs_predicates.cuh"

namespace cs {

int bits_tensor_map(CUtensorMap *map, const uint64_t *base, int64_t B, int64_t N, int64_t stride, int box_bytes, int rows,
                    bool swizzle64);      // cs_interval_pair.cu

namespace {

constexpr int TCT = 256;                 // tile edge (pairs): two M = 128 accumulators of 256 columns
constexpr int TC_EPI_WARPS = 16;
constexpr int TC_EPI0 = 2;               // warp 0: loader, warp 1: MMA issuer + TMEM owner, warps 2..17: epilogue,
constexpr int TC_WR0 = TC_EPI0 + TC_EPI_WARPS;   // warps 18..19: writers (staged tile -> global memory)
constexpr int TC_WR_WARPS = 2;
constexpr int TC_THREADS = (TC_WR0 + TC_WR_WARPS) * 32;
constexpr int TC_PITCH = 9;              // words per staged row (8 + 1: conflict-free 4-byte stores by 32 rows)
constexpr int TC_NF = 12;                // columns of a 32 x 32 block whose sign bit goes through the FMA pipe (0 .. 23)

// Per-point data of the tensor route: Fast<> of cs_predicates.cuh for the predicates cs_build.cu already treats as
// bilinear forms, and two more that are bilinear in derived coordinates only.  F_c is component fcomp(c) of the point's
// vector (P_c is component c, negated for c < NNEG); time() is what the tiles must be ordered by.
template <int GEOM, int DIM>
struct TcFast : Fast<GEOM, DIM> {
    static constexpr bool RANGE2 = false;        // the tile also needs a bounded range of the second coordinate
    __device__ static __forceinline__ double time(const double *x) { return x[0]; }
    __device__ static __forceinline__ constexpr int fcomp(int c) { return c; }
};
// 1+1 light cone: (u_i < u_j) && (v_i < v_j)  <=>  T = du dv > 0 and du + dv > 0;  T = h_i + h_j - u_i v_j - v_i u_j with
// h = u v.  Tiles ordered by t = (u + v) / 2: a pair decided "related" has |du dv| > m, far more than the rounding of t, so
// du + dv > 0 follows from t_j >= t_i and both differences are positive.
template <>
struct TcFast<CS_GEOM_MINK2_LIGHTCONE, 2> {
    static constexpr bool H = true, RANGE2 = false, STRICT = false;
    static constexpr int NP = 2, NNEG = 2, MARGIN = 64;
    __device__ static __forceinline__ double time(const double *x) { return (x[0] + x[1]) * 0.5; }
    __device__ static __forceinline__ constexpr int fcomp(int c) { return 1 - c; }
    __device__ static __forceinline__ bool convert(const double *x, float *v, float &h)
    {
        v[0] = (float)x[0];
        v[1] = (float)x[1];
        h = (float)(x[0] * x[1]);
        return true;
    }
};
// 1+1 de Sitter slab: with omega = min(|dtheta|, 2 pi - |dtheta|) the arc between the two angles and 0 <= d eta <= pi,
// d eta >= omega  <=>  T = cos(dtheta) - cos(d eta) >= 0, bilinear in (cos eta, sin eta, cos theta, sin theta) formed per
// point in fp64.  The header's expression is that arc only while |dtheta| <= 2 pi: a tile takes the band only if its angles
// span at most 2 pi and its times at most pi (RANGE2); the fp64 rows use the header's expression as everywhere.
template <>
struct TcFast<CS_GEOM_DS2_SLAB, 2> {
    static constexpr bool H = false, RANGE2 = true, STRICT = false;
    static constexpr int NP = 4, NNEG = 2, MARGIN = 64;
    __device__ static __forceinline__ double time(const double *x) { return x[0]; }
    __device__ static __forceinline__ constexpr int fcomp(int c) { return c; }
    __device__ static __forceinline__ bool convert(const double *x, float *v, float &h)
    {
        double s0, c0, s1, c1;
        sincos(x[0], &s0, &c0);
        sincos(x[1], &s1, &c1);
        v[0] = (float)c0; v[1] = (float)s0; v[2] = (float)c1; v[3] = (float)s1;
        h = 0.f;
        return isfinite(x[0]) && isfinite(x[1]);
    }
};

template <int GEOM, int DIM>
struct TcShape {
    using F = TcFast<GEOM, DIM>;
    static constexpr int USED = 6 * F::NP + (F::H ? 6 : 2);     // without h two columns carry the padding marker
    static constexpr int K = USED <= 32 ? 32 : 48;
    static constexpr int KC = K / 8;                              // 16-byte chunks per operand row
    static constexpr int A_BLOCK = KC * 128 * 16;                 // operand image of 128 past points
    static constexpr int B_BLOCK = KC * 256 * 16;                 // operand image of 256 future points
    static constexpr int STAGE = 2 * A_BLOCK + B_BLOCK;
    static_assert(USED <= 48, "operand columns");
};

struct TcBlockInfo {                     // summary of 128 consecutive points
    double tmin, tmax;                   // over the valid points (+inf / -inf if none)
    float C;                             // largest |fp32 component|
    uint32_t flags;                      // 1: t non-decreasing inside the block, 2: last point <= first of the next block, 4: a point
                                         // that may not use the prefilter (not finite, or Fast::convert says no)
    float cmax[6];                       // largest |fp32 component| per component (0 beyond NP)
    float hmax;                          // largest |h|
    float x1min, x1max;                  // range of the second coordinate, rounded outwards (RANGE2 geometries only)
    uint32_t pad;
};
static_assert(sizeof(TcBlockInfo) == 64, "TcBlockInfo");

__device__ __forceinline__ uint32_t tc_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void tc_mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(tc_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void tc_mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc_smem_u32(bar)) : "memory");
}
// try_wait with a suspend-time hint: the thread sleeps in hardware until the phase completes (or the hint expires)
// instead of spinning through issue slots the epilogue warps need
__device__ __forceinline__ void tc_mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra LAB_DONE;\n"
        "bra LAB_WAIT;\n"
        "LAB_DONE:\n"
        "}\n" ::"r"(tc_smem_u32(bar)),
        "r"(parity), "r"(0x989680u)
        : "memory");
}
// the same for the roles that mostly wait (loader, MMA issuer, writers): between two tries the warp sleeps, so that its
// polling does not take issue slots from the epilogue warps of its scheduler (12 % of all instructions without it)
__device__ __forceinline__ void tc_mbar_wait_sleep(uint64_t *bar, uint32_t parity, uint32_t ns)
{
    uint32_t done;
    while (true) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(tc_smem_u32(bar)), "r"(parity), "r"(0x989680u) : "memory");
        if (done) break;
        __nanosleep(ns);
    }
}
__device__ __forceinline__ void tc_mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tc_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tc_bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     tc_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(tc_smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// shared-memory matrix descriptor: no swizzle, K-major; LBO = distance between 16-byte k chunks, SBO = between
// groups of 8 rows (both in bytes); bit 46 = descriptor version of sm_100
__device__ __forceinline__ uint64_t tc_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// instruction descriptor, kind::f16: D = F32 (1 at bit 4), A = B = BF16 (1 at bits 7 and 10), both K-major,
// N >> 3 at bit 17, M >> 4 at bit 24
constexpr uint32_t TC_IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(256 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

__device__ __forceinline__ void tc_mma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t accum)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(TC_IDESC), "r"(accum)
        : "memory");
}
__device__ __forceinline__ void tc_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(tc_smem_u32(bar))
                 : "memory");
}
// 32 lanes x 32 columns -> 32 registers per thread; the caller issues tcgen05.wait::ld
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t *v)
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

// v = hi + mid + lo exactly (each piece rounded to nearest; 24 significand bits = 3 x 8)
__device__ __forceinline__ void split3(float v, uint16_t (&p)[3])
{
    const __nv_bfloat16 a = __float2bfloat16_rn(v);
    const float r1 = v - __bfloat162float(a);
    const __nv_bfloat16 b = __float2bfloat16_rn(r1);
    const float r2 = r1 - __bfloat162float(b);
    const __nv_bfloat16 c = __float2bfloat16_rn(r2);
    p[0] = __bfloat16_as_ushort(a);
    p[1] = __bfloat16_as_ushort(b);
    p[2] = __bfloat16_as_ushort(c);
}

// ---- prep: one thread per point ------------------------------------------------------------------
// Operand columns, in this order (pairs (A column of the past point, B column of the future point)):
//   rank 0:  (P_hi, F_hi) per component                      [+ (h_hi, 1), (1, h_hi)]
//   rank 1:  (P_hi, F_mid), (P_mid, F_hi) per component      [+ (h_mid, 1), (1, h_mid)]
//   rank 2:  (P_mid, F_mid), (P_hi, F_lo), (P_lo, F_hi)      [+ (h_lo, 1), (1, h_lo)]
// A point beyond N has zero components and h = -2^100 (exactly one bf16 piece), so that every pair it belongs to reads
// a = -2^100 or -2^101: "unrelated", far outside the band.  Predicates without h carry the marker in two columns of
// their own, (pad, 1) and (1, pad), pad = 0 for a valid point.
constexpr float TC_PAD = -0x1p100f;

template <int GEOM, int DIM>
__global__ void __launch_bounds__(128)
k_tc_prep(const double *__restrict__ coords, int64_t N, int nA,
          unsigned char *__restrict__ opA, unsigned char *__restrict__ opB, TcBlockInfo *__restrict__ info,
          double *__restrict__ cpad)
{
    using F = TcFast<GEOM, DIM>;
    using S = TcShape<GEOM, DIM>;
    constexpr int NP = F::NP;
    const int a = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t b = blockIdx.y;
    coords += b * N * DIM;
    const int64_t gp = (int64_t)a * 128 + tid;
    const bool valid = gp < N;

    double x[DIM];
#pragma unroll
    for (int d = 0; d < DIM; d++) x[d] = valid ? coords[gp * DIM + d] : 0.0;
    {   // padded copy of the coordinates (NaN beyond N: unrelated to everything) for the fp64 rows of the main kernel
        const double qnan = __longlong_as_double(0x7FF8000000000000LL);
        double *cp = cpad + (((size_t)b * nA + a) * 128 + tid) * DIM;
#pragma unroll
        for (int d = 0; d < DIM; d++) cp[d] = valid ? x[d] : qnan;
    }
    float v[NP], h = 0.f;
    bool ok = F::convert(x, v, h);
    float c = 0.f;
#pragma unroll
    for (int q = 0; q < NP; q++) {
        c = fmaxf(c, fabsf(v[q]));
        ok = ok && isfinite(v[q]);
    }
    ok = ok && isfinite(h) && isfinite(F::time(x));       // a NaN time would slip through the fmin / fmax of the block summary
    if (!valid) {
#pragma unroll
        for (int q = 0; q < NP; q++) v[q] = 0.f;
        h = F::H ? TC_PAD : 0.f;
        c = 0.f;
        ok = true;
    }

    // operand rows
    uint16_t A[S::K], Bv[S::K];
    {
        uint16_t P[NP][3], Fp[NP][3], hp[3], pp[3];
#pragma unroll
        for (int q = 0; q < NP; q++) {
            split3(v[F::fcomp(q)], Fp[q]);
            split3(q < F::NNEG ? -v[q] : v[q], P[q]);
        }
        split3(h, hp);
        split3(valid ? 0.f : TC_PAD, pp);
        constexpr uint16_t ONE = 0x3F80;
        int k = 0;
#pragma unroll
        for (int q = 0; q < NP; q++) { A[k] = P[q][0]; Bv[k] = Fp[q][0]; k++; }
        if (F::H) { A[k] = hp[0]; Bv[k] = ONE; k++; A[k] = ONE; Bv[k] = hp[0]; k++; }
        else      { A[k] = pp[0]; Bv[k] = ONE; k++; A[k] = ONE; Bv[k] = pp[0]; k++; }
#pragma unroll
        for (int q = 0; q < NP; q++) {
            A[k] = P[q][0]; Bv[k] = Fp[q][1]; k++;
            A[k] = P[q][1]; Bv[k] = Fp[q][0]; k++;
        }
        if (F::H) { A[k] = hp[1]; Bv[k] = ONE; k++; A[k] = ONE; Bv[k] = hp[1]; k++; }
#pragma unroll
        for (int q = 0; q < NP; q++) {
            A[k] = P[q][1]; Bv[k] = Fp[q][1]; k++;
            A[k] = P[q][0]; Bv[k] = Fp[q][2]; k++;
            A[k] = P[q][2]; Bv[k] = Fp[q][0]; k++;
        }
        if (F::H) { A[k] = hp[2]; Bv[k] = ONE; k++; A[k] = ONE; Bv[k] = hp[2]; k++; }
#pragma unroll
        for (; k < S::K; k++) { A[k] = 0; Bv[k] = 0; }
    }
    unsigned char *dA = opA + ((size_t)b * nA + a) * S::A_BLOCK + (size_t)tid * 16;
    unsigned char *dB = opB + ((size_t)b * (nA / 2) + (a >> 1)) * S::B_BLOCK + (size_t)((a & 1) * 128 + tid) * 16;
#pragma unroll
    for (int kc = 0; kc < S::KC; kc++) {
        uint4 wa, wb;
        wa.x = A[8 * kc] | ((uint32_t)A[8 * kc + 1] << 16);
        wa.y = A[8 * kc + 2] | ((uint32_t)A[8 * kc + 3] << 16);
        wa.z = A[8 * kc + 4] | ((uint32_t)A[8 * kc + 5] << 16);
        wa.w = A[8 * kc + 6] | ((uint32_t)A[8 * kc + 7] << 16);
        wb.x = Bv[8 * kc] | ((uint32_t)Bv[8 * kc + 1] << 16);
        wb.y = Bv[8 * kc + 2] | ((uint32_t)Bv[8 * kc + 3] << 16);
        wb.z = Bv[8 * kc + 4] | ((uint32_t)Bv[8 * kc + 5] << 16);
        wb.w = Bv[8 * kc + 6] | ((uint32_t)Bv[8 * kc + 7] << 16);
        *reinterpret_cast<uint4 *>(dA + (size_t)kc * 128 * 16) = wa;
        *reinterpret_cast<uint4 *>(dB + (size_t)kc * 256 * 16) = wb;
    }

    // block summary
    const double inf = __longlong_as_double(0x7FF0000000000000LL);
    const double tp = F::time(x);
    double tmn = valid ? tp : inf, tmx = valid ? tp : -inf;
    bool sorted = true;                                   // this point <= the next one (fp64; NaN: false)
    if (valid && gp + 1 < N) {                            // F::STRICT: the time is not part of T, d eta > 0 comes from the order alone
        const double tn = F::time(coords + (gp + 1) * DIM);
        sorted = F::STRICT ? tp < tn : tp <= tn;
    }
    float x1lo = __int_as_float(0x7f800000), x1hi = __int_as_float(0xff800000);
    if (F::RANGE2 && valid) { x1lo = __double2float_rd(x[1]); x1hi = __double2float_ru(x[1]); }
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        tmn = fmin(tmn, __shfl_xor_sync(0xffffffffu, tmn, s));
        tmx = fmax(tmx, __shfl_xor_sync(0xffffffffu, tmx, s));
        c = fmaxf(c, __shfl_xor_sync(0xffffffffu, c, s));
        if (F::RANGE2) {
            x1lo = fminf(x1lo, __shfl_xor_sync(0xffffffffu, x1lo, s));
            x1hi = fmaxf(x1hi, __shfl_xor_sync(0xffffffffu, x1hi, s));
        }
    }
    __shared__ double s_mn[4], s_mx[4];
    __shared__ float s_c[4], s_x1[4][2];
    __shared__ uint32_t s_cm[4][7];
    uint32_t cm[7];                                       // |component| and |h| maxima: non-negative floats order like their bits
#pragma unroll
    for (int q = 0; q < 6; q++) cm[q] = __reduce_max_sync(0xffffffffu, (q < NP && valid) ? (__float_as_uint(v[q]) & 0x7fffffffu) : 0u);
    cm[6] = __reduce_max_sync(0xffffffffu, (F::H && valid) ? (__float_as_uint(h) & 0x7fffffffu) : 0u);
    if (lane == 0) {
        s_mn[warp] = tmn; s_mx[warp] = tmx; s_c[warp] = c;
        s_x1[warp][0] = x1lo; s_x1[warp][1] = x1hi;
#pragma unroll
        for (int q = 0; q < 7; q++) s_cm[warp][q] = cm[q];
    }
    const int inner = __syncthreads_and(sorted || tid == 127);
    const int link = __syncthreads_and(sorted || tid != 127);
    const int bad = __syncthreads_or(!ok);
    if (tid == 0) {
        TcBlockInfo bi;
        bi.tmin = fmin(fmin(s_mn[0], s_mn[1]), fmin(s_mn[2], s_mn[3]));
        bi.tmax = fmax(fmax(s_mx[0], s_mx[1]), fmax(s_mx[2], s_mx[3]));
        bi.C = fmaxf(fmaxf(s_c[0], s_c[1]), fmaxf(s_c[2], s_c[3]));
        bi.flags = (inner ? 1u : 0u) | (link ? 2u : 0u) | (bad ? 4u : 0u);
#pragma unroll
        for (int q = 0; q < 6; q++) bi.cmax[q] = __uint_as_float(max(max(s_cm[0][q], s_cm[1][q]), max(s_cm[2][q], s_cm[3][q])));
        bi.hmax = __uint_as_float(max(max(s_cm[0][6], s_cm[1][6]), max(s_cm[2][6], s_cm[3][6])));
        if (F::fcomp(0) != 0) {                       // P_c and F_c are different components: one bound for all products
#pragma unroll
            for (int q = 0; q < 6; q++) bi.cmax[q] = q < NP ? bi.C : 0.f;
        }
        bi.x1min = fminf(fminf(s_x1[0][0], s_x1[1][0]), fminf(s_x1[2][0], s_x1[3][0]));
        bi.x1max = fmaxf(fmaxf(s_x1[0][1], s_x1[1][1]), fmaxf(s_x1[2][1], s_x1[3][1]));
        bi.pad = 0;
        info[(size_t)b * nA + a] = bi;
    }
}

// ---- tile table ------------------------------------------------------------------------------------
// One entry per tile of the launch, row-major over the upper triangle (J >= I) of every causet:
//   x = I | J << 16, y = causet, z = margin m (float bits; +inf: every row of the tile goes to fp64), w = unused.
__global__ void __launch_bounds__(256)
k_tc_tiles(const TcBlockInfo *__restrict__ info, int nT, uint32_t tiles_per, uint32_t total_tiles, float acc_units,
           float in_units, int range2, int strict, uint4 *__restrict__ tab)
{
    const uint32_t t = blockIdx.x * 256 + threadIdx.x;
    if (t >= total_tiles) return;
    const uint32_t b = t / tiles_per, idx = t - b * tiles_per;
    const double w = 2.0 * nT + 1.0;
    int I = (int)((w - sqrt(w * w - 8.0 * (double)idx)) * 0.5);
    if (I < 0) I = 0;
    if (I > nT - 1) I = nT - 1;
    auto off = [&](int r) { return (uint32_t)r * (uint32_t)nT - (uint32_t)((int64_t)r * (r - 1) / 2); };
    while (I > 0 && off(I) > idx) I--;
    while (I + 1 < nT && off(I + 1) <= idx) I++;
    const int J = I + (int)(idx - off(I));
    const TcBlockInfo *bi = info + (size_t)b * 2 * nT;
    const TcBlockInfo i0 = bi[2 * I], i1 = bi[2 * I + 1], j0 = bi[2 * J], j1 = bi[2 * J + 1];
    const float C = fmaxf(fmaxf(i0.C, i1.C), fmaxf(j0.C, j1.C));
    const bool bad = ((i0.flags | i1.flags | j0.flags | j1.flags) & 4u) != 0;
    const bool ordered = (I == J) ? ((i0.flags & 3u) == 3u && (i1.flags & 1u) != 0)
                                  : (strict ? fmax(i0.tmax, i1.tmax) < fmin(j0.tmin, j1.tmin)
                                            : fmax(i0.tmax, i1.tmax) <= fmin(j0.tmin, j1.tmin));
    bool fast = !bad && ordered && C >= 0x1p-40f && C <= 0x1p40f;
    if (range2) {       // 1+1 dS slab: times within pi and angles within 2 pi over the whole tile (both tested a little short)
        const double tspan = fmax(j0.tmax, j1.tmax) - fmin(i0.tmin, i1.tmin);
        const float aspan = __fsub_ru(fmaxf(fmaxf(i0.x1max, i1.x1max), fmaxf(j0.x1max, j1.x1max)),
                                      fminf(fminf(i0.x1min, i1.x1min), fminf(j0.x1min, j1.x1min)));
        fast = fast && tspan <= 3.1415926 && aspan <= 6.2831845f;
    }
    // largest single addend a pair of this tile can hand to the tensor core: |h_i|, |h_j|, |P_c(i) F_c(j)|
    float M = fmaxf(fmaxf(i0.hmax, i1.hmax), fmaxf(j0.hmax, j1.hmax));
#pragma unroll
    for (int q = 0; q < 6; q++) M = fmaxf(M, __fmul_ru(fmaxf(i0.cmax[q], i1.cmax[q]), fmaxf(j0.cmax[q], j1.cmax[q])));
    const float m = fast ? __fmul_ru(1.001f * 0x1p-24f, __fmaf_ru(acc_units, M, __fmul_ru(in_units, __fmul_ru(C, C))))
                         : __int_as_float(0x7f800000);
    tab[t] = make_uint4((uint32_t)I | ((uint32_t)J << 16), b, __float_as_uint(m), __float_as_uint(C));
}

// ---- main kernel -----------------------------------------------------------------------------------
struct TcProbe {                 // cs_a1_tensor_probe: what the prefilter saw (all tiles of the launch)
    unsigned int max_err_bits;   // max |a - T| / C^2 as float bits (pairs decided by sign)
    unsigned int max_acc_bits;   // max |a - exact sum of the operand products| / C^2: the tensor core's own accumulation error
    unsigned int max_ratio_bits; // max |a - T| / m, m = the margin of the pair's tile: must stay below 1
    unsigned int pad;
    unsigned long long rows_fp64;   // (row, 32-column block) pairs re-evaluated in fp64
    unsigned long long rows_total;  // (row, block) pairs examined
};

template <int GEOM, int DIM>
struct TcSmem {
    using S = TcShape<GEOM, DIM>;
    static constexpr int NSTG = S::K == 32 ? 3 : 2;                 // operand stages (one tile each)
    static constexpr int COORD = TCT * DIM * 8;                     // fp64 coordinates of 256 points (for the fp64 rows)
    static constexpr int STAGE = S::STAGE + 2 * COORD;              // [A 2 blocks][B][coords I][coords J]
    static constexpr size_t STAGING = (size_t)NSTG * STAGE;         // uint32 [2][256][TC_PITCH] x 2 (U, L)
    static constexpr size_t ZERO = STAGING + 4 * TCT * TC_PITCH * 4;   // 256 x 32 bytes of zeros (source of the mirrored tiles)
    static constexpr size_t BARS = ZERO + TCT * 32;
    static constexpr size_t BYTES = BARS + (2 * NSTG + 8) * 8 + 16;
    static_assert(STAGE % 16 == 0 && BYTES <= 227 * 1024, "k_causal_tc: shared memory");
};

template <int GEOM, int DIM, bool PROBE>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_causal_tc(const __grid_constant__ CUtensorMap mapB, const __grid_constant__ CUtensorMap mapT,
            const double *__restrict__ cpad, const unsigned char *__restrict__ opA,
            const unsigned char *__restrict__ opB, const uint4 *__restrict__ tab,
            int64_t N, int64_t stride, int nT, uint32_t total_tiles,
            uint64_t *__restrict__ bits, uint64_t *__restrict__ bitsT, TcProbe *__restrict__ probe)
{
    using S = TcShape<GEOM, DIM>;
    using SM = TcSmem<GEOM, DIM>;
    constexpr int NSTG = SM::NSTG;
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *s_stage = smem;
    uint32_t *s_U = reinterpret_cast<uint32_t *>(smem + SM::STAGING);                    // [2][256][TC_PITCH]
    uint32_t *s_L = s_U + 2 * TCT * TC_PITCH;                                            // [2][256][TC_PITCH]
    uint64_t *s_full = reinterpret_cast<uint64_t *>(smem + SM::BARS);                    // [NSTG] operands landed
    uint64_t *s_empty = s_full + NSTG;                                                   // [NSTG] stage free again
    uint64_t *s_tfull = s_empty + NSTG;                                                  // [2] accumulator complete
    uint64_t *s_tempty = s_tfull + 2;                                                    // [2] accumulator drained
    uint64_t *s_sfull = s_tempty + 2;                                                    // [2] staged tile complete
    uint64_t *s_sempty = s_sfull + 2;                                                    // [2] staged tile written out
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(s_sempty + 2);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nA = 2 * nT;

    if (tid == 0) {
        for (int s = 0; s < NSTG; s++) {
            tc_mbar_init(&s_full[s], 1);
            tc_mbar_init(&s_empty[s], 1 + TC_EPI_WARPS);      // the MMAs (commit) and every epilogue warp (fp64 rows read the coordinates)
        }
        for (int h = 0; h < 2; h++) {
            tc_mbar_init(&s_tfull[h], 1);
            tc_mbar_init(&s_tempty[h], TC_EPI_WARPS);
            tc_mbar_init(&s_sfull[h], TC_EPI_WARPS);
            tc_mbar_init(&s_sempty[h], TC_WR_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < TCT * 32 / 16; i += TC_THREADS) reinterpret_cast<uint4 *>(smem + SM::ZERO)[i] = make_uint4(0, 0, 0, 0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // read by TMA stores
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(tc_smem_u32(s_tmem)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *s_tmem;

    if (warp == 0) {
        // ===================================== loader =========================================
        if (lane == 0) {
            uint32_t n = 0;
            for (uint32_t t = blockIdx.x; t < total_tiles; t += gridDim.x, n++) {
                const uint4 e = __ldg(tab + t);
                const uint32_t I = e.x & 0xFFFFu, J = e.x >> 16, b = e.y;
                const uint32_t s = n % NSTG;
                tc_mbar_wait_sleep(&s_empty[s], ((n / NSTG) & 1) ^ 1, 800);
                tc_mbar_expect_tx(&s_full[s], (uint32_t)SM::STAGE);
                unsigned char *dst = s_stage + (size_t)s * SM::STAGE;
                const unsigned char *cp = reinterpret_cast<const unsigned char *>(cpad) + (size_t)b * nT * SM::COORD;
                tc_bulk_g2s(dst, opA + ((size_t)b * nA + 2 * I) * S::A_BLOCK, 2 * S::A_BLOCK, &s_full[s]);
                tc_bulk_g2s(dst + 2 * S::A_BLOCK, opB + ((size_t)b * nT + J) * S::B_BLOCK, S::B_BLOCK, &s_full[s]);
                tc_bulk_g2s(dst + S::STAGE, cp + (size_t)I * SM::COORD, SM::COORD, &s_full[s]);
                tc_bulk_g2s(dst + S::STAGE + SM::COORD, cp + (size_t)J * SM::COORD, SM::COORD, &s_full[s]);
            }
        }
    } else if (warp == 1) {
        // ===================================== MMA issuer =====================================
        if (lane == 0) {
            uint32_t n = 0;
            for (uint32_t t = blockIdx.x; t < total_tiles; t += gridDim.x, n++) {
                const uint32_t s = n % NSTG;
                tc_mbar_wait_sleep(&s_full[s], (n / NSTG) & 1, 100);
                const uint32_t a_addr = tc_smem_u32(s_stage + (size_t)s * SM::STAGE);
                const uint32_t b_addr = a_addr + 2 * S::A_BLOCK;
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    tc_mbar_wait_sleep(&s_tempty[h], (n & 1) ^ 1, 100);     // the epilogue has read accumulator h of the tile before
                    tc_fence_after();
#pragma unroll
                    for (int q = 0; q < S::KC / 2; q++) {             // K = 16 per instruction: two 16-byte chunks
                        const uint64_t ad = tc_desc(a_addr + h * S::A_BLOCK + q * 2 * 128 * 16, 128 * 16, 128);
                        const uint64_t bd = tc_desc(b_addr + q * 2 * 256 * 16, 256 * 16, 128);
                        tc_mma_bf16(tmem_base + h * 256, ad, bd, q > 0 ? 1u : 0u);
                    }
                    tc_commit(&s_tfull[h]);
                }
                tc_commit(&s_empty[s]);
            }
        }
    } else if (warp < TC_WR0) {
        // ===================================== epilogue =======================================
        const int e = warp - TC_EPI0;
        const int q = warp & 3;                       // TMEM lane quarter this warp may read
        const int g = e >> 2;                         // 64 columns of the 256
        const TransposeLane transpose(lane);
        uint32_t n = 0;
        float p_err = 0.f, p_acc = 0.f, p_ratio = 0.f;
        unsigned long long p_rows = 0, p_tot = 0;
        uint2 ent = blockIdx.x < total_tiles ? __ldg(reinterpret_cast<const uint2 *>(tab + blockIdx.x)) : make_uint2(0, 0);
        uint32_t ent_m = blockIdx.x < total_tiles ? __ldg(reinterpret_cast<const uint32_t *>(tab + blockIdx.x) + 2) : 0;
        for (uint32_t t = blockIdx.x; t < total_tiles; t += gridDim.x, n++) {
            const bool diag = (ent.x & 0xFFFFu) == (ent.x >> 16);
            const float m = __uint_as_float(ent_m);
            float C2 = 0.f;
            if (PROBE) {
                const float C = __uint_as_float(__ldg(reinterpret_cast<const uint32_t *>(tab + t) + 3));
                C2 = C * C;
            }
            if (t + gridDim.x < total_tiles) {                     // next tile's entry, a tile ahead
                ent = __ldg(reinterpret_cast<const uint2 *>(tab + t + gridDim.x));
                ent_m = __ldg(reinterpret_cast<const uint32_t *>(tab + t + gridDim.x) + 2);
            }
            const uint32_t s = n % NSTG;
            const double *cI = reinterpret_cast<const double *>(s_stage + (size_t)s * SM::STAGE + S::STAGE);
            const double *cJ = cI + TCT * DIM;
            uint32_t *U = s_U + (n & 1) * TCT * TC_PITCH, *L = s_L + (n & 1) * TCT * TC_PITCH;
            tc_mbar_wait(&s_sempty[n & 1], ((n >> 1) & 1) ^ 1);    // the writers are done with this staging buffer
            tc_mbar_wait(&s_full[s], (n / NSTG) & 1);              // the stage's coordinates (read by the fp64 rows) have landed:
                                                                   // complete long before, but this is the wait that orders the reads

            // The blocks of a tile are software-pipelined: the shuffle butterfly of the block before (five dependent
            // shuffles, ~150 clk of latency) is interleaved with the sign extraction of the current one.
            auto do_tile = [&](auto diag_tag) {
                constexpr bool DIAG = decltype(diag_tag)::value;
                uint32_t pend = 0;                    // word of the block before, not yet transposed
                uint32_t *pendL = L + lane * TC_PITCH;   // where its transpose goes (first use: a dummy store of 0, overwritten)
                bool have = false;
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int r0 = h * 128 + q * 32;                  // first row of this warp's blocks (tile-local)
                    tc_mbar_wait(&s_tfull[h], n & 1);
                    tc_fence_after();
                    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + h * 256 + g * 64;
#pragma unroll
                    for (int k = 0; k < 2; k++) {
                        const int c0 = g * 64 + k * 32;               // first column of the block (tile-local)
                        uint32_t lw = 0;
                        if (DIAG && c0 + 31 <= r0) {                  // a block at or below the diagonal: all zero
                            if (have) *pendL = transpose(pend);
                            U[(r0 + lane) * TC_PITCH + (c0 >> 5)] = 0;
                            pend = 0;
                            pendL = L + (c0 + lane) * TC_PITCH + (r0 >> 5);
                            have = true;
                            continue;
                        }
                        uint32_t v[32];
                        tc_ld32(taddr + k * 32, v);
                        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                        if (DIAG && c0 == r0) {                       // the block on the diagonal: T(i, i) = 0 would send every row
#pragma unroll
                            for (int c = 0; c < 32; c++)              // to fp64; pairs with j <= i read -inf (unrelated, outside the band)
                                if (c <= lane) v[c] = 0xff800000u;
                        }
                        // Sign bits.  The kernel is bound by instruction issue and by the ALU pipe (SHF, FMNMX3, LOP3: one warp
                        // instruction per two clocks) while the FMA pipe is idle: TC_NF columns take their bit through it,
                        //     t = fma.sat(a, 2^100, 0.5)      1.0 if a > 0, 0.0 if a < 0 (|a| > m >= 2^-94; in-band rows are redone)
                        //     acc = fma(t, 2^c, acc)           acc = 2^23 + sum: the bits sit in the significand
                        // (two FMA-pipe instructions per pair) and the others through the funnel shift (one ALU instruction per
                        // pair); TC_NF balances the two pipes against the issue slots.  min |a| over all 32 columns stays on the
                        // ALU pipe (one FMNMX3 per two pairs, two independent chains).  The five butterfly steps of the block
                        // before are spread between them by hand (ptxas keeps the shuffles together otherwise).
                        uint32_t sg = 0;
                        float acc = 0x1p23f;
                        float mn0 = __int_as_float(0x7f800000), mn1 = mn0;
                        uint32_t px = pend, po;
#define TC_BIT(c)                                                                                           \
    if ((c) < TC_NF) {                                                                                      \
        float t_;                                                                                           \
        asm("fma.rn.sat.f32 %0, %1, 0f71800000, 0f3F000000;" : "=f"(t_) : "f"(__uint_as_float(v[c])));      \
        acc = __fmaf_rn(t_, (float)(1u << ((c) < TC_NF ? (c) : 0)), acc);                                   \
    } else {                                                                                                \
        sg = __funnelshift_l(v[c], sg, 1);                                                                  \
    }
#define TC_MIN(c)                                                      \
    mn0 = min3_abs_nan(mn0, v[c], v[c - 1]);                           \
    mn1 = min3_abs_nan(mn1, v[16 + c], v[16 + c - 1]);
#define TC_BFLY_SEND(t) po = __shfl_xor_sync(0xffffffffu, px, 16 >> t);
#define TC_BFLY_TAKE(t)                                                \
    po = __funnelshift_l(po, po, transpose.rot[t]);                    \
    px = (px & transpose.keep[t]) | (po & ~transpose.keep[t]);
                        TC_BFLY_SEND(0)
                        TC_BIT(31) TC_BIT(30) TC_BIT(0) TC_BIT(29) TC_BIT(28) TC_BIT(1) TC_BIT(27)
                        TC_MIN(15) TC_MIN(13)
                        TC_BFLY_TAKE(0) TC_BFLY_SEND(1)
                        TC_BIT(26) TC_BIT(2) TC_BIT(25) TC_BIT(24) TC_BIT(3) TC_BIT(23) TC_BIT(22)
                        TC_MIN(11) TC_MIN(9)
                        TC_BFLY_TAKE(1) TC_BFLY_SEND(2)
                        TC_BIT(4) TC_BIT(21) TC_BIT(20) TC_BIT(5) TC_BIT(19) TC_BIT(18) TC_BIT(6)
                        TC_MIN(7) TC_MIN(5)
                        TC_BFLY_TAKE(2) TC_BFLY_SEND(3)
                        TC_BIT(17) TC_BIT(16) TC_BIT(7) TC_BIT(15) TC_BIT(14) TC_BIT(13)
                        TC_MIN(3)
                        TC_BFLY_TAKE(3) TC_BFLY_SEND(4)
                        TC_BIT(12) TC_BIT(11) TC_BIT(10) TC_BIT(9) TC_BIT(8)
                        TC_MIN(1)
                        TC_BFLY_TAKE(4)
#undef TC_BIT
#undef TC_MIN
#undef TC_BFLY_SEND
#undef TC_BFLY_TAKE
                        const uint32_t pendT = px;
                        // bits 0..NF-1: related = 1, from the significand of acc (0x4B000000 | bits); the other columns: related =
                        // sign clear, sg holds their signs (column 31 highest):  lw = bits + ((2^(32-NF) - 1 - sg) << NF)
                        lw = (__float_as_uint(acc) - 0x4B000000u + (0xFFFFFFFFu << TC_NF)) - (sg << TC_NF);
                        const bool unc = !(mn0 > m && mn1 > m);       // NaN compares false: uncertain
                        uint32_t todo = __ballot_sync(0xffffffffu, unc);
                        if (have) *pendL = pendT;                     // past of j: bit = row i
                        if (PROBE) {
                            p_tot++;
                            p_rows += unc ? 1 : 0;
                            if (GEOM == CS_GEOM_MINK_CONE && !unc) {
#pragma unroll
                                for (int c = 0; c < 32; c++) {
                                    double T = 0.0;
#pragma unroll
                                    for (int d = 0; d < DIM; d++) {
                                        const double dd = cJ[(c0 + c) * DIM + d] - cI[(r0 + lane) * DIM + d];
                                        T += d == 0 ? dd * dd : -dd * dd;
                                    }
                                    const float er = (float)(fabs((double)__uint_as_float(v[c]) - 0.5 * T) / (double)C2);
                                    if (er == er && isfinite(__uint_as_float(v[c]))) {      // (padding points are NaN, masked pairs -inf)
                                        p_err = fmaxf(p_err, er);
                                        p_ratio = fmaxf(p_ratio, er * C2 / m);
                                    }
                                    // the same pair from the operand rows the tensor core read (every product of two bf16
                                    // pieces is exact in fp64, and so is their sum to 2^-50)
                                    const unsigned char *st_ = s_stage + (size_t)s * SM::STAGE;
                                    const int ra = (r0 + lane) & 127, hb = (r0 + lane) >> 7;
                                    double ex = 0.0;
                                    for (int kk = 0; kk < S::K; kk++) {
                                        const uint16_t ua = *reinterpret_cast<const uint16_t *>(
                                            st_ + hb * S::A_BLOCK + ((kk >> 3) * 128 + ra) * 16 + (kk & 7) * 2);
                                        const uint16_t ub = *reinterpret_cast<const uint16_t *>(
                                            st_ + 2 * S::A_BLOCK + ((kk >> 3) * 256 + c0 + c) * 16 + (kk & 7) * 2);
                                        ex += (double)__uint_as_float((uint32_t)ua << 16) * (double)__uint_as_float((uint32_t)ub << 16);
                                    }
                                    const float ea = (float)(fabs((double)__uint_as_float(v[c]) - ex) / (double)C2);
                                    if (er == er && fabs(ex) < 1e30 && isfinite(__uint_as_float(v[c]))) p_acc = fmaxf(p_acc, ea);
                                }
                            }
                        }
                        while (todo) {                                // fp64 for whole rows of the block, one pair per lane
                            const int r = __ffs(todo) - 1;
                            todo &= todo - 1;
                            double xi[DIM], xj[DIM];
#pragma unroll
                            for (int d = 0; d < DIM; d++) {
                                xi[d] = cI[(r0 + r) * DIM + d];       // (points beyond N are NaN: unrelated)
                                xj[d] = cJ[(c0 + lane) * DIM + d];
                            }
                            const uint32_t w = __ballot_sync(0xffffffffu, Pred<GEOM, DIM>::rel(xi, xj));
                            if (lane == r) lw = w;
                        }
                        if (DIAG) {                                   // only i < j inside the diagonal tile
                            const int keep_from = r0 + lane + 1 - c0;              // columns c >= keep_from are kept
                            lw &= keep_from <= 0 ? 0xffffffffu : (keep_from >= 32 ? 0u : (0xffffffffu << keep_from));
                        }
                        U[(r0 + lane) * TC_PITCH + (c0 >> 5)] = lw;                   // future of i: bit = column j
                        pend = lw;
                        pendL = L + (c0 + lane) * TC_PITCH + (r0 >> 5);
                        have = true;
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) tc_mbar_arrive(&s_tempty[h]);      // accumulator h may be overwritten
                }
                *pendL = transpose(pend);
            };
            if (diag) do_tile(std::true_type{});
            else do_tile(std::false_type{});
            __syncwarp();
            if (lane == 0) {
                tc_mbar_arrive(&s_empty[s]);          // this warp no longer reads the stage's coordinates
                tc_mbar_arrive(&s_sfull[n & 1]);      // its part of the staged tile is complete
            }
        }
        if (PROBE) {
#pragma unroll
            for (int sft = 16; sft >= 1; sft >>= 1) {
                p_err = fmaxf(p_err, __shfl_xor_sync(0xffffffffu, p_err, sft));
                p_acc = fmaxf(p_acc, __shfl_xor_sync(0xffffffffu, p_acc, sft));
                p_ratio = fmaxf(p_ratio, __shfl_xor_sync(0xffffffffu, p_ratio, sft));
                p_rows += __shfl_xor_sync(0xffffffffu, p_rows, sft);
                p_tot += __shfl_xor_sync(0xffffffffu, p_tot, sft);
            }
            if (lane == 0) {
                atomicMax(&probe->max_err_bits, __float_as_uint(p_err));
                atomicMax(&probe->max_acc_bits, __float_as_uint(p_acc));
                atomicMax(&probe->max_ratio_bits, __float_as_uint(p_ratio));
                atomicAdd(&probe->rows_fp64, p_rows);
                atomicAdd(&probe->rows_total, p_tot);
            }
        }
    } else {
        // ===================================== writers ========================================
        // 64 threads move a staged tile to global memory: thread = (row mod 32, 16-byte half of the 32-byte segment),
        // eight rows each.  The mirrored tile of an off-diagonal tile is zeros: two TMA tile stores from a constant zero
        // tile (rows beyond N and bytes beyond the row are clipped by the tensor map).
        const int wt = tid - TC_WR0 * 32;             // 0 .. 63
        const int hf = wt & 1, rr = wt >> 1;
        const int64_t row_bytes = stride * 8;
        uint32_t n = 0;
        for (uint32_t t = blockIdx.x; t < total_tiles; t += gridDim.x, n++) {
            const uint4 e = __ldg(tab + t);
            const int I = (int)(e.x & 0xFFFFu), J = (int)(e.x >> 16);
            if (wt == 0 && I != J) {
                const uint32_t zsrc = tc_smem_u32(smem + SM::ZERO);
                asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(&mapB),
                             "r"(I * 32), "r"(J * TCT), "r"((int)e.y), "r"(zsrc) : "memory");
                if (bitsT)
                    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(&mapT),
                                 "r"(J * 32), "r"(I * TCT), "r"((int)e.y), "r"(zsrc) : "memory");
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
            const int64_t colI = (int64_t)I * 32 + hf * 16, colJ = (int64_t)J * 32 + hf * 16;      // byte offsets in a row
            const size_t mat = (size_t)e.y * N * row_bytes;
            unsigned char *pb = reinterpret_cast<unsigned char *>(bits) + mat + colJ;
            unsigned char *pt = reinterpret_cast<unsigned char *>(bitsT) + mat + colI;
            const bool okI = colI < row_bytes && bitsT != nullptr, okJ = colJ < row_bytes;
            const uint32_t *u = s_U + (n & 1) * TCT * TC_PITCH + rr * TC_PITCH + hf * 4;
            const uint32_t *l = s_L + (n & 1) * TCT * TC_PITCH + rr * TC_PITCH + hf * 4;
            int64_t gi = (int64_t)I * TCT + rr, gj = (int64_t)J * TCT + rr;
            tc_mbar_wait_sleep(&s_sfull[n & 1], (n >> 1) & 1, 400);
#pragma unroll
            for (int p = 0; p < 8; p++) {
                if (gi < N && okJ) *reinterpret_cast<uint4 *>(pb + (size_t)gi * row_bytes) = make_uint4(u[0], u[1], u[2], u[3]);
                if (gj < N && okI) *reinterpret_cast<uint4 *>(pt + (size_t)gj * row_bytes) = make_uint4(l[0], l[1], l[2], l[3]);
                u += 32 * TC_PITCH;
                l += 32 * TC_PITCH;
                gi += 32;
                gj += 32;
            }
            __syncwarp();
            if (lane == 0) tc_mbar_arrive(&s_sempty[n & 1]);
        }
        if (wt == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base));
    }
}

template <int GEOM, int DIM>
size_t tc_scratch_t(int64_t B, int64_t N)
{
    using S = TcShape<GEOM, DIM>;
    const size_t nT = (size_t)((N + TCT - 1) / TCT);
    const size_t tiles = (size_t)B * (nT * (nT + 1) / 2);
    return align_up((size_t)B * 2 * nT * S::A_BLOCK, 256) + align_up((size_t)B * nT * S::B_BLOCK, 256) +
           align_up((size_t)B * 2 * nT * sizeof(TcBlockInfo), 256) + align_up((size_t)B * nT * TCT * DIM * 8, 256) +
           align_up(tiles * sizeof(uint4), 256);
}

template <int GEOM, int DIM, bool PROBE>
int launch_tc_t(const double *coords, int64_t B, int64_t N, int64_t stride, uint64_t *bits, uint64_t *bitsT,
                void *scratch, TcProbe *probe, cudaStream_t st)
{
    using S = TcShape<GEOM, DIM>;
    const int nT = (int)((N + TCT - 1) / TCT);
    const int64_t tiles_per = (int64_t)nT * (nT + 1) / 2;
    if (nT > 32768 || B > 65535 || tiles_per * B >= ((int64_t)1 << 32)) return CS_ERR_ARG;
    using SM = TcSmem<GEOM, DIM>;
    const int64_t total = tiles_per * B;
    unsigned char *opA = static_cast<unsigned char *>(scratch);
    unsigned char *opB = opA + align_up((size_t)B * 2 * nT * S::A_BLOCK, 256);
    TcBlockInfo *info = reinterpret_cast<TcBlockInfo *>(opB + align_up((size_t)B * nT * S::B_BLOCK, 256));
    double *cpad = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(info) + align_up((size_t)B * 2 * nT * sizeof(TcBlockInfo), 256));
    uint4 *tab = reinterpret_cast<uint4 *>(reinterpret_cast<unsigned char *>(cpad) + align_up((size_t)B * nT * TCT * DIM * 8, 256));
    k_tc_prep<GEOM, DIM><<<dim3(2 * nT, (unsigned)B), 128, 0, st>>>(coords, N, 2 * nT, opA, opB, info, cpad);
    CS_LAUNCHED("k_tc_prep");
    // margin m = (ACC M + IN C^2) 2^-24, see the header: ACC = 4 (K + 2) (twice the alignment loss of K + 2 addends),
    // IN = the fp32 prefilter's own bound (Fast::MARGIN / 2, conversions included) + the dropped piece products
    k_tc_tiles<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(info, nT, (uint32_t)tiles_per, (uint32_t)total,
                                                                 4.f * (S::K + 2), (float)(TcFast<GEOM, DIM>::MARGIN / 2 + 3 * TcFast<GEOM, DIM>::NP),
                                                                 TcFast<GEOM, DIM>::RANGE2 ? 1 : 0, TcFast<GEOM, DIM>::STRICT ? 1 : 0, tab);
    CS_LAUNCHED("k_tc_tiles");
    constexpr size_t smem = SM::BYTES;
    static PerDeviceFlag attr_set;
    const int dev = current_device();
    if (!attr_set.get(dev)) {
        CS_CUDA(cudaFuncSetAttribute(k_causal_tc<GEOM, DIM, PROBE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set.set(dev);
    }
    CUtensorMap mapB, mapT;
    int rc = bits_tensor_map(&mapB, bits, B, N, stride, 32, TCT, false);
    if (rc) return rc;
    rc = bits_tensor_map(&mapT, bitsT ? bitsT : bits, B, N, stride, 32, TCT, false);
    if (rc) return rc;
    int grid = sm_count();
    if (grid > total) grid = (int)total;
    k_causal_tc<GEOM, DIM, PROBE><<<grid, TC_THREADS, smem, st>>>(mapB, mapT, cpad, opA, opB, tab, N, stride, nT, (uint32_t)total,
                                                                  bits, bitsT, probe);
    CS_LAUNCHED("k_causal_tc");
    return CS_OK;
}

}  // namespace

bool causal_tc_supported(int geometry, int dim)
{
    if (!interval_tensor_available()) return false;      // (a constant true: the library is built for sm_100a only)
    switch (geometry) {
    case CS_GEOM_MINK2_LIGHTCONE: return dim == 2;
    case CS_GEOM_DS2_SLAB: return dim == 2;
    case CS_GEOM_MINK_CONE: return dim >= 2 && dim <= 5;
    case CS_GEOM_FLRW_POLAR: return dim == 6;
    case CS_GEOM_DS4_SPHERICAL: return dim == 7;
    default: return false;
    }
}

#define CS_TC_DISPATCH(CALL)                                                                       \
    switch (geometry) {                                                                            \
    case CS_GEOM_MINK2_LIGHTCONE:                                                                  \
        if (dim == 2) return CALL(CS_GEOM_MINK2_LIGHTCONE, 2);                                     \
        break;                                                                                     \
    case CS_GEOM_DS2_SLAB:                                                                         \
        if (dim == 2) return CALL(CS_GEOM_DS2_SLAB, 2);                                            \
        break;                                                                                     \
    case CS_GEOM_MINK_CONE:                                                                        \
        if (dim == 2) return CALL(CS_GEOM_MINK_CONE, 2);                                           \
        if (dim == 3) return CALL(CS_GEOM_MINK_CONE, 3);                                           \
        if (dim == 4) return CALL(CS_GEOM_MINK_CONE, 4);                                           \
        if (dim == 5) return CALL(CS_GEOM_MINK_CONE, 5);                                           \
        break;                                                                                     \
    case CS_GEOM_FLRW_POLAR:                                                                       \
        if (dim == 6) return CALL(CS_GEOM_FLRW_POLAR, 6);                                          \
        break;                                                                                     \
    case CS_GEOM_DS4_SPHERICAL:                                                                    \
        if (dim == 7) return CALL(CS_GEOM_DS4_SPHERICAL, 7);                                       \
        break;                                                                                     \
    default:                                                                                       \
        break;                                                                                     \
    }

size_t causal_tc_scratch_bytes(int64_t B, int64_t N, int dim, int geometry)
{
#define CS_TC_SCRATCH(G, D) tc_scratch_t<G, D>(B, N)
    CS_TC_DISPATCH(CS_TC_SCRATCH)
#undef CS_TC_SCRATCH
    return 0;
}

int launch_causal_tc(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                     uint64_t *bits, uint64_t *bitsT, void *scratch, cudaStream_t st)
{
    const int64_t stride = row_stride_words(N);
#define CS_TC_LAUNCH(G, D) launch_tc_t<G, D, false>(coords, B, N, stride, bits, bitsT, scratch, nullptr, st)
    CS_TC_DISPATCH(CS_TC_LAUNCH)
#undef CS_TC_LAUNCH
    return CS_ERR_GEOM;
}

// The same launch with the probe counters switched on (flat cone in 3+1 and 4+1 dimensions: K = 32 and K = 48).
// out_host: [0] largest |a - T| / (2^-24 C^2) over the pairs decided by sign, [1] (row, block) pairs sent to fp64,
// [2] (row, block) pairs examined, [3] largest |a - T| / m with m the margin of the pair's tile (< 1 or a decision by sign
// could be wrong), [4] largest |a - exact sum of the operand products|
// in the same unit (what the tensor core's accumulation alone lost).
int launch_causal_tc_probe(const double *coords, int64_t N, int dim, uint64_t *bits, uint64_t *bitsT,
                           void *scratch, double *out_host, cudaStream_t st)
{
    const int64_t stride = row_stride_words(N);
    TcProbe *dp = nullptr;
    CS_CUDA(cudaMallocAsync(reinterpret_cast<void **>(&dp), sizeof(TcProbe), st));
    TcProbe hp;
    memset(&hp, 0, sizeof(hp));
    // every exit below passes the cudaFreeAsync: the counters are not leaked when a step fails
    int rc = [&]() -> int {
        CS_CUDA(cudaMemsetAsync(dp, 0, sizeof(TcProbe), st));
        int r = CS_ERR_DIM;
        if (dim == 4) r = launch_tc_t<CS_GEOM_MINK_CONE, 4, true>(coords, 1, N, stride, bits, bitsT, scratch, dp, st);
        if (dim == 5) r = launch_tc_t<CS_GEOM_MINK_CONE, 5, true>(coords, 1, N, stride, bits, bitsT, scratch, dp, st);
        if (r) return r;
        CS_CUDA(cudaMemcpyAsync(&hp, dp, sizeof(hp), cudaMemcpyDeviceToHost, st));
        CS_CUDA(cudaStreamSynchronize(st));
        return CS_OK;
    }();
    cudaFreeAsync(dp, st);
    if (rc) return rc;
    float err;
    memcpy(&err, &hp.max_err_bits, 4);
    out_host[0] = (double)err * 16777216.0;
    out_host[1] = (double)hp.rows_fp64;
    out_host[2] = (double)hp.rows_total;
    memcpy(&err, &hp.max_ratio_bits, 4);
    out_host[3] = (double)err;
    memcpy(&err, &hp.max_acc_bits, 4);
    out_host[4] = (double)err * 16777216.0;
    return CS_OK;
}

}  // namespace cs
