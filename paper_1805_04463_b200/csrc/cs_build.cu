// cs_build.cu -- stage a1: causal-matrix build, plus the
// bit-matrix transpose and the relation statistics (R, W_alg).
//
// One CTA owns one BT x BT tile (I <= J) of the pair space.  The BT "past" points x_i of the
// tile are staged in shared memory (the paper's Alg. 16 idea, for both
// elements: PAPER.md:1695); every lane keeps one "future" point x_j in registers and sweeps
// 32 rows at a time.  The predicate is evaluated ONCE per pair and yields both outputs:
//   bits  (row i, bit j)  through a warp ballot     -> "future of i"
//   bitsT (row j, bit i)  accumulated in the lane   -> "past of j"
// Both tiles are assembled in shared memory and written with full 32-byte row segments.
// The same CTA zero-fills the mirrored tile (lower triangle), so no separate memset is needed.
//
// Floating point: explicit round-to-nearest intrinsics (__dsub_rn, __dmul_rn, __dadd_rn), which
// the compiler never contracts into FMA, in exactly the order stated in include/causalset.h.
#include <atomic>
#include <mutex>

#include "cs_predicates.cuh"

namespace cs {

constexpr int BT = 256;          // tile edge in elements
constexpr int BUILD_THREADS = 256;


// order-preserving map float -> uint32 (NaN with the sign bit clear sorts above +inf, set below -inf)
__device__ __forceinline__ uint32_t float_key(float f)
{
    const uint32_t u = __float_as_uint(f);
    return u ^ ((uint32_t)((int32_t)u >> 31) | 0x80000000u);
}
__device__ __forceinline__ float key_float(uint32_t k)
{
    return __uint_as_float(k ^ ((k & 0x80000000u) ? 0x80000000u : 0xFFFFFFFFu));
}

constexpr int NJ = 2;            // future points per lane: a CTA covers 256 rows x 512 columns

// Packed single precision (Blackwell FFMA2 / FADD2: two fp32 lanes per instruction, each rounded like the scalar
// operation, so the error bound above is unchanged).  A 64-bit register holds the values of two consecutive rows.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 bcast2(float v)
{
    f32x2 d;
    asm("mov.b64 %0, {%1, %1};" : "=l"(d) : "f"(v));     // ptxas folds this into the .F32 broadcast operand form
    return d;
}
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 fmul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 fadd2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
// One 32 x 32 block per future point k < NK of this lane: bit ii of lw[k] = (row i0 + ii  -<  point k),
// decided by the fp32 prefilter; unc[k] is set if any of the lane's 32 decisions is inside the error
// band (or NaN).
//
// Bilinear forms (flat cone, FLRW, 3+1 de Sitter): the past points sit in shared memory as NP (+1) arrays
// (-t, x, y, z, h for the 3+1 cone), so one LDS.128 brings a component of four consecutive rows and each 64-bit half feeds a packed operation on two rows; the future
// point's coordinates are per-lane scalars that FFMA2 broadcasts.  Per four pairs: 8 FFMA2 + 2 FADD2 for the
// values, then one SHF per pair shifts the value's sign bit into the lane's word and one FMNMX3 per two pairs
// keeps the smallest |a| -- if that exceeds the margin m, no decision of the block is inside the band, and
// "a > m" is simply "sign bit clear".  4 instructions per pair instead of 8 (4 FFMA, FADD, 2 FSETP, predicated add).
template <int GEOM, int DIM, int NK>
__device__ __forceinline__ void fast_block(const float *__restrict__ sf, int i0,
                                           const float (*fj)[Fast<GEOM, DIM>::NP], const float *hj, const float *m,
                                           uint32_t *lw, bool *unc)
{
    constexpr int NP = Fast<GEOM, DIM>::NP;
    constexpr bool H = Fast<GEOM, DIM>::H;
    if (GEOM == CS_GEOM_DS2_SLAB) {
        const float2 *fi = reinterpret_cast<const float2 *>(sf) + i0;     // (eta, theta) per past point
#pragma unroll
        for (int ii = 0; ii < 32; ii++) {
            const float2 p = fi[ii];
#pragma unroll
            for (int k = 0; k < NK; k++) {
                const float de = fj[k][0] - p.x;
                const float ab = fabsf(fj[k][1] - p.y);
                const float a = de - fminf(ab, 6.2831853071795865f - ab);
                if (a > m[k]) lw[k] |= 1u << ii;
                unc[k] = unc[k] || !(fabsf(a) > m[k]);
            }
        }
        return;
    }
    uint32_t sg[NK];
    float mn[NK];
    f32x2 fb[NK][NP], fh[NK];
#pragma unroll
    for (int k = 0; k < NK; k++) {
        sg[k] = 0;
        mn[k] = __int_as_float(0x7f800000);
#pragma unroll
        for (int c = 0; c < NP; c++) fb[k][c] = bcast2(fj[k][c]);
        fh[k] = bcast2(hj[k]);
    }
#pragma unroll
    for (int i4 = 0; i4 < 32; i4 += 4) {
        ulonglong2 P[NP], Hh;                           // component c of rows (0,1), (2,3)
#pragma unroll
        for (int c = 0; c < NP; c++) P[c] = *reinterpret_cast<const ulonglong2 *>(sf + c * BT + i0 + i4);
        if (H) Hh = *reinterpret_cast<const ulonglong2 *>(sf + NP * BT + i0 + i4);
#pragma unroll
        for (int k = 0; k < NK; k++) {
            f32x2 a01, a23;
            if (H) {
                a01 = ffma2(P[0].x, fb[k][0], Hh.x);
                a23 = ffma2(P[0].y, fb[k][0], Hh.y);
            } else {
                a01 = fmul2(P[0].x, fb[k][0]);
                a23 = fmul2(P[0].y, fb[k][0]);
            }
#pragma unroll
            for (int c = 1; c < NP; c++) {
                a01 = ffma2(P[c].x, fb[k][c], a01);
                a23 = ffma2(P[c].y, fb[k][c], a23);
            }
            if (H) {
                a01 = fadd2(a01, fh[k]);
                a23 = fadd2(a23, fh[k]);
            }
            const uint32_t a0 = (uint32_t)a01, a1 = (uint32_t)(a01 >> 32), a2 = (uint32_t)a23, a3 = (uint32_t)(a23 >> 32);
            sg[k] = __funnelshift_l(a0, sg[k], 1);      // row i0 + ii ends up at bit 31 - ii
            sg[k] = __funnelshift_l(a1, sg[k], 1);
            sg[k] = __funnelshift_l(a2, sg[k], 1);
            sg[k] = __funnelshift_l(a3, sg[k], 1);
            mn[k] = min3_abs_nan(mn[k], a0, a1);
            mn[k] = min3_abs_nan(mn[k], a2, a3);
        }
    }
#pragma unroll
    for (int k = 0; k < NK; k++) {
        lw[k] = ~__brev(sg[k]);              // related = sign bit clear (valid when no decision is inside the band)
        unc[k] = !(mn[k] > m[k]);            // NaN compares false: uncertain
    }
}

// The same block with the fp64 expression of include/causalset.h (the definition).
template <int GEOM, int DIM, int NK>
__device__ __forceinline__ void exact_block(const double (*xi_s)[BT], int i0, const double (*xj)[DIM], uint32_t *lw)
{
#pragma unroll 8
    for (int ii = 0; ii < 32; ii++) {
        double xi[DIM];
#pragma unroll
        for (int d = 0; d < DIM; d++) xi[d] = xi_s[d][i0 + ii];
#pragma unroll
        for (int k = 0; k < NK; k++) lw[k] |= (Pred<GEOM, DIM>::rel(xi, xj[k]) ? 1u : 0u) << ii;
    }
}

// shared memory of one CTA (dynamic: the wider geometries pass the 48 KB static limit)
template <int GEOM, int DIM>
struct BuildSmem {
    using F = Fast<GEOM, DIM>;
    static constexpr int NF = F::ok ? F::NP + (F::H ? 1 : 0) : 0;          // fp32 arrays of the past points
    static constexpr size_t XI = 0;                                         // double [DIM][BT]
    static constexpr size_t SF = XI + (size_t)DIM * BT * 8;                 // float  [NF][BT]
    static constexpr size_t SU = SF + (size_t)NF * BT * 4;                  // uint32 [BT][NJ * 8 + 1]
    static constexpr size_t SL = SU + (size_t)BT * (NJ * 8 + 1) * 4;        // uint32 [NJ * BT][9]
    static constexpr size_t BYTES = SL + (size_t)NJ * BT * 9 * 4;
    static_assert(SF % 16 == 0 && SU % 16 == 0 && BYTES <= 56 * 1024, "k_causal_matrix: shared memory (four CTAs per SM)");
};

template <int GEOM, int DIM>
__global__ void __launch_bounds__(BUILD_THREADS)
k_causal_matrix(const double *__restrict__ coords, int64_t N, int64_t stride,
                uint64_t *__restrict__ bits, uint64_t *__restrict__ bitsT)
{
    const int JS = blockIdx.x, I = blockIdx.y;
    const int nT = gridDim.y;
    if (JS * NJ + NJ - 1 < I) return;             // every column tile of this CTA lies below the diagonal
    const int64_t b = blockIdx.z;
    coords += b * N * DIM;
    bits += b * N * stride;
    if (bitsT) bitsT += b * N * stride;

    using F = Fast<GEOM, DIM>;
    using SM = BuildSmem<GEOM, DIM>;
    constexpr bool FAST = F::ok;
    constexpr int NP = F::NP;
    constexpr int NW = BUILD_THREADS / 32;
    extern __shared__ __align__(16) unsigned char dsm[];
    double (*s_xi)[BT] = reinterpret_cast<double (*)[BT]>(dsm + SM::XI);
    // fp32 copies of the past points: NP component arrays (+ h); dS slab: (eta, theta) pairs
    float *s_f = reinterpret_cast<float *>(dsm + SM::SF);
    uint32_t (*s_U)[NJ * 8 + 1] = reinterpret_cast<uint32_t (*)[NJ * 8 + 1]>(dsm + SM::SU);   // row i_local, word = 32 columns j
    uint32_t (*s_L)[9] = reinterpret_cast<uint32_t (*)[9]>(dsm + SM::SL);                     // row j_local, word = 32 rows i
    uint32_t (*s_red)[NW] = reinterpret_cast<uint32_t (*)[NW]>(dsm + SM::SU);   // [2 + 2 NJ][NW], dead before s_U is written

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double qnan = __longlong_as_double(0x7FF8000000000000LL);   // compares false: unrelated
    const int jl = warp * 32 + lane;

    const TransposeLane transpose(lane);
    bool act[NJ], dg[NJ];
    bool any_diag = false;
#pragma unroll
    for (int k = 0; k < NJ; k++) {
        const int J = JS * NJ + k;
        act[k] = J >= I && J < nT;
        dg[k] = J == I;
        any_diag = any_diag || dg[k];
    }

    double xi0[DIM];
    {   // stage the tile's past points (SoA), NaN beyond N
        int64_t gi = (int64_t)I * BT + tid;
#pragma unroll
        for (int d = 0; d < DIM; d++) {
            xi0[d] = (gi < N) ? coords[gi * DIM + d] : qnan;
            s_xi[d][tid] = xi0[d];
        }
    }
    double xj[NJ][DIM];
#pragma unroll
    for (int k = 0; k < NJ; k++) {
        int64_t gj = (int64_t)(JS * NJ + k) * BT + jl;
#pragma unroll
        for (int d = 0; d < DIM; d++) xj[k][d] = (act[k] && gj < N) ? coords[gj * DIM + d] : qnan;
    }

    bool fast[NJ];
    float fj[NJ][NP], hj[NJ], m[NJ];
#pragma unroll
    for (int k = 0; k < NJ; k++) {
        fast[k] = false; hj[k] = 0.f; m[k] = 0.f;
#pragma unroll
        for (int c = 0; c < NP; c++) fj[k][c] = 0.f;
    }
    if (FAST) {
        // Tile summaries, all as floats reduced with redux.sync on order-preserving integer keys:
        //   C   >= largest |component| of the past points and of each set of future points (the fp32
        //          conversions, NaN ignored by fmaxf; rounding to nearest is covered by m's 1.001); a point that
        //          may not use the prefilter (Fast::convert) reports +inf, which fails the range test below,
        //   max t_i rounded up and min t_j rounded down, so "max t_i <= min t_j" is only ever claimed when
        //   it holds for the doubles (a NaN time makes the claim fail or is ignored: safe where the time is part of
        //   T, and where it is not -- F::STRICT -- convert() has already refused the point).
        // Inside the diagonal tile i < j must imply t_i <= t_j instead: its points are in time order.
        // F::STRICT: both claims with < (the header's expression wants d eta > 0 and T does not see eta).
        float fi[NP], hi0, ci = 0.f;
        const bool oki = F::convert(xi0, fi, hi0);
#pragma unroll
        for (int c = 0; c < NP; c++) ci = fmaxf(ci, fabsf(fi[c]));
        // a real point that may not use the prefilter takes the tile off it (padding beyond N is NaN and harmless)
        if (!oki && (int64_t)I * BT + tid < N) ci = __int_as_float(0x7f800000);
        if (GEOM == CS_GEOM_DS2_SLAB) {
            reinterpret_cast<float2 *>(s_f)[tid] = make_float2(fi[0], fi[1]);
        } else {
#pragma unroll
            for (int c = 0; c < NP; c++) s_f[c * BT + tid] = c < F::NNEG ? -fi[c] : fi[c];
            if (F::H) s_f[NP * BT + tid] = hi0;
        }
        const uint32_t wci = __reduce_max_sync(0xffffffffu, __float_as_uint(ci));   // ci >= 0: bit order = value order
        const uint32_t wti = __reduce_max_sync(0xffffffffu, float_key(__double2float_ru(xi0[0])));
        if (lane == 0) { s_red[0][warp] = wci; s_red[1][warp] = wti; }
#pragma unroll
        for (int k = 0; k < NJ; k++) {
            float cj = 0.f;
            const bool okj = F::convert(xj[k], fj[k], hj[k]);
#pragma unroll
            for (int c = 0; c < NP; c++) cj = fmaxf(cj, fabsf(fj[k][c]));
            if (!okj && act[k] && (int64_t)(JS * NJ + k) * BT + jl < N) cj = __int_as_float(0x7f800000);
            const uint32_t wcj = __reduce_max_sync(0xffffffffu, __float_as_uint(cj));
            const uint32_t wtj = __reduce_max_sync(0xffffffffu, float_key(-__double2float_rd(xj[k][0])));   // -(min t_j)
            if (lane == 0) { s_red[2 + 2 * k][warp] = wcj; s_red[3 + 2 * k][warp] = wtj; }
        }
        __syncthreads();
        uint32_t r[2 + 2 * NJ];
#pragma unroll
        for (int q = 0; q < 2 + 2 * NJ; q++) {
            r[q] = s_red[q][0];
#pragma unroll
            for (int w = 1; w < NW; w++) r[q] = max(r[q], s_red[q][w]);
        }
        bool tile_ordered = false;
        if (any_diag) {   // points beyond N are NaN and only ever sit at the end: their pairs read unrelated either way
            const bool last = tid == BT - 1 || (int64_t)I * BT + tid + 1 >= N;
            const double tnext = s_xi[0][last ? tid : tid + 1];
            tile_ordered = __syncthreads_and(last || (F::STRICT ? xi0[0] < tnext : xi0[0] <= tnext)) != 0;
        }
        const float Ci = __uint_as_float(r[0]), tmaxI = key_float(r[1]);
#pragma unroll
        for (int k = 0; k < NJ; k++) {
            const float C = fmaxf(Ci, __uint_as_float(r[2 + 2 * k]));
            if (GEOM == CS_GEOM_DS2_SLAB) {
                const float Cd = fmaxf(C, 6.2831855f);                     // >= 2 pi
                fast[k] = act[k] && (Cd <= 0x1p100f);
                m[k] = __fmul_ru(Cd, 0x1p-19f * 1.001f);
            } else {
                const float tminJ = -key_float(r[3 + 2 * k]);
                const bool ordered = dg[k] ? tile_ordered : (F::STRICT ? tmaxI < tminJ : tmaxI <= tminJ);
                fast[k] = act[k] && ordered && (C >= 0x1p-40f) && (C <= 0x1p40f);
                m[k] = __fmul_ru(__fmul_ru(C, C), (float)F::MARGIN * 0x1p-24f * 1.001f);
            }
        }
    }
    __syncthreads();    // s_xi / s_f visible; s_red (aliased on s_U) no longer read

    // The common CTA -- both column tiles above the diagonal and on the prefilter -- runs a loop with nothing in it
    // but the blocks, the (rare) fp64 fallback, the two transposes and four shared-memory stores; everything that
    // depends on diagonal tiles, inactive tiles or tiles off the prefilter stays in the general loop below.
    const bool plain = FAST && !any_diag && act[0] && act[1] && fast[0] && fast[1];
    if (plain) {
        uint32_t *pL0 = &s_L[jl][0], *pL1 = &s_L[BT + jl][0], *pU = &s_U[lane][warp];
#pragma unroll 1
        for (int sb = 0; sb < BT / 32; sb++) {
            uint32_t lw[NJ] = {0, 0};
            bool unc[NJ] = {false, false};
            fast_block<GEOM, DIM, 2>(s_f, sb * 32, fj, hj, m, lw, unc);
            if (__any_sync(0xffffffffu, unc[0] || unc[1])) {
                lw[0] = lw[1] = 0;
                exact_block<GEOM, DIM, 2>(s_xi, sb * 32, xj, lw);
            }
            pL0[sb] = lw[0];
            pL1[sb] = lw[1];
            pU[sb * 32 * (NJ * 8 + 1)] = transpose(lw[0]);
            pU[sb * 32 * (NJ * 8 + 1) + 8] = transpose(lw[1]);
        }
    }
#pragma unroll 1
    for (int sb = plain ? BT / 32 : 0; sb < BT / 32; sb++) {
        uint32_t lw[NJ];
        bool need[NJ], slow[NJ];
#pragma unroll
        for (int k = 0; k < NJ; k++) {
            lw[k] = 0;
            need[k] = act[k] && !(dg[k] && sb > warp);   // rows all at or below the diagonal: nothing to evaluate
            slow[k] = need[k] && !fast[k];
        }
        if (FAST) {
            bool unc[NJ] = {false, false};
            const bool f0 = need[0] && fast[0], f1 = need[1] && fast[1];
            if (f0 && f1) fast_block<GEOM, DIM, 2>(s_f, sb * 32, fj, hj, m, lw, unc);
            else if (f0) fast_block<GEOM, DIM, 1>(s_f, sb * 32, fj, hj, m, lw, unc);
            else if (f1) fast_block<GEOM, DIM, 1>(s_f, sb * 32, fj + 1, hj + 1, m + 1, lw + 1, unc + 1);
#pragma unroll
            for (int k = 0; k < NJ; k++) {
                if (__any_sync(0xffffffffu, unc[k])) { slow[k] = true; lw[k] = 0; }
            }
        }
        if (slow[0] && slow[1]) exact_block<GEOM, DIM, 2>(s_xi, sb * 32, xj, lw);
        else if (slow[0]) exact_block<GEOM, DIM, 1>(s_xi, sb * 32, xj, lw);
        else if (slow[1]) exact_block<GEOM, DIM, 1>(s_xi, sb * 32, xj + 1, lw + 1);
#pragma unroll
        for (int k = 0; k < NJ; k++) {
            if (dg[k]) {   // only i < j inside the diagonal tile
                const int lo = jl - sb * 32;   // rows sb*32 + ii with ii < lo are kept
                lw[k] &= lo <= 0 ? 0u : (lo >= 32 ? 0xffffffffu : ((1u << lo) - 1u));
            }
            if (act[k]) {
                s_L[k * BT + jl][sb] = lw[k];                                   // past of j: bit = row i
                s_U[sb * 32 + lane][k * 8 + warp] = transpose(lw[k]);   // future of i: bit = column j
            }
        }
    }
    __syncthreads();

    // write-out.  Rows of the I tile: NJ x 4 uint64 per row, 8 consecutive threads cover one 64-byte segment
    // (bits: the tile; bitsT: zeros, the mirrored tile of an off-diagonal tile is identically zero).
    {
        const int q8 = tid & 7, k = q8 >> 2, q = q8 & 3;
        const int J = JS * NJ + k;
        const int64_t wj = (int64_t)J * (BT / 64) + q;
        if (J >= I && J < nT && wj < stride) {
#pragma unroll
            for (int pass = 0; pass < 8; pass++) {
                const int r = (tid >> 3) + 32 * pass;
                const int64_t ri = (int64_t)I * BT + r;
                if (ri < N) {
                    bits[ri * stride + wj] = (uint64_t)s_U[r][k * 8 + 2 * q] | ((uint64_t)s_U[r][k * 8 + 2 * q + 1] << 32);
                    if (bitsT && J != I) bitsT[ri * stride + wj] = 0;
                }
            }
        }
    }
    // Rows of the J tiles: 4 uint64 per row, 4 consecutive threads cover one 32-byte segment
    {
        const int q = tid & 3;
        const int64_t wi = (int64_t)I * (BT / 64) + q;
        if (wi < stride) {
#pragma unroll
            for (int pass = 0; pass < NJ * 4; pass++) {
                const int r2 = (tid >> 2) + 64 * pass;          // 0 .. NJ*256-1
                const int k = r2 / BT, r = r2 % BT;
                const int J = JS * NJ + k;
                const int64_t rj = (int64_t)J * BT + r;
                if (J >= I && J < nT && rj < N) {
                    if (bitsT) bitsT[rj * stride + wi] = (uint64_t)s_L[r2][2 * q] | ((uint64_t)s_L[r2][2 * q + 1] << 32);
                    if (J != I) bits[rj * stride + wi] = 0;
                }
            }
        }
    }
}

// Columns of the last tile may stop short of the row stride (stride is rounded up to an even
// word count); those padding words are zeroed here.
__global__ void k_zero_tail(uint64_t *bits, uint64_t *bitsT, int64_t rows, int64_t stride, int64_t first_word)
{
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= rows) return;
    for (int64_t w = first_word; w < stride; w++) {
        bits[r * stride + w] = 0;
        if (bitsT) bitsT[r * stride + w] = 0;
    }
}

template <int GEOM, int DIM>
static int launch_build_t(const double *coords, int64_t B, int64_t N, int64_t stride,
                          uint64_t *bits, uint64_t *bitsT, cudaStream_t st)
{
    const int nT = (int)((N + BT - 1) / BT);
    dim3 grid((nT + NJ - 1) / NJ, nT, (unsigned)B);   // x: groups of NJ column tiles, y: row tile
    constexpr size_t smem = BuildSmem<GEOM, DIM>::BYTES;
    if (smem > 48 * 1024) {
        static PerDeviceFlag attr_set;
        const int dev = current_device();
        if (!attr_set.get(dev)) {
            CS_CUDA(cudaFuncSetAttribute(k_causal_matrix<GEOM, DIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            attr_set.set(dev);
        }
    }
    k_causal_matrix<GEOM, DIM><<<grid, BUILD_THREADS, smem, st>>>(coords, N, stride, bits, bitsT);
    CS_LAUNCHED("k_causal_matrix");
    const int64_t covered = (int64_t)nT * (BT / 64);
    if (covered < stride) {
        int64_t rows = B * N;
        k_zero_tail<<<(unsigned)((rows + 255) / 256), 256, 0, st>>>(bits, bitsT, rows, stride, covered);
        CS_LAUNCHED("k_zero_tail");
    }
    return CS_OK;
}

static int launch_causal_fma(const double *coords, int64_t B, int64_t N, int dim, int geometry,
                             uint64_t *bits, uint64_t *bitsT, cudaStream_t st)
{
    const int64_t stride = row_stride_words(N);
    if (N > (int64_t)BT * 65535 || B > 65535) return CS_ERR_ARG;
    switch (geometry) {
    case CS_GEOM_MINK2_LIGHTCONE:
        if (dim != 2) return CS_ERR_DIM;
        return launch_build_t<CS_GEOM_MINK2_LIGHTCONE, 2>(coords, B, N, stride, bits, bitsT, st);
    case CS_GEOM_MINK_CONE:
        if (dim == 2) return launch_build_t<CS_GEOM_MINK_CONE, 2>(coords, B, N, stride, bits, bitsT, st);
        if (dim == 3) return launch_build_t<CS_GEOM_MINK_CONE, 3>(coords, B, N, stride, bits, bitsT, st);
        if (dim == 4) return launch_build_t<CS_GEOM_MINK_CONE, 4>(coords, B, N, stride, bits, bitsT, st);
        if (dim == 5) return launch_build_t<CS_GEOM_MINK_CONE, 5>(coords, B, N, stride, bits, bitsT, st);
        return CS_ERR_DIM;
    case CS_GEOM_DS2_SLAB:
        if (dim != 2) return CS_ERR_DIM;
        return launch_build_t<CS_GEOM_DS2_SLAB, 2>(coords, B, N, stride, bits, bitsT, st);
    case CS_GEOM_FLRW_POLAR:
        if (dim != 6) return CS_ERR_DIM;
        return launch_build_t<CS_GEOM_FLRW_POLAR, 6>(coords, B, N, stride, bits, bitsT, st);
    case CS_GEOM_DS4_SPHERICAL:
        if (dim != 7) return CS_ERR_DIM;
        return launch_build_t<CS_GEOM_DS4_SPHERICAL, 7>(coords, B, N, stride, bits, bitsT, st);
    default:
        return CS_ERR_GEOM;
    }
}

// Which kernel builds the matrix.  The tensor route (cs_build_tc.cu) serves the bilinear predicates; it is a persistent
// kernel over 256 x 256 tiles, one CTA per SM, and wins once there are about as many tiles as SMs (measured on B200,
// flat cone in 3+1: 0.38 against 0.75 ms at N = 65536, 0.043 against 0.071 ms at N = 16384; a single causet of N = 2048 --
// 36 tiles -- takes 0.034 against 0.023 ms, while 296 of them take 0.13 against 0.27 ms).
constexpr int64_t TC_MIN_TILES = 128;

static int resolve_a1_route(int64_t B, int64_t N, int dim, int geometry, int route)
{
    if (route == CS_A1_FMA) return CS_A1_FMA;
    const bool can = causal_tc_supported(geometry, dim) && N >= 256;      // (rows of at least 32 bytes: TMA boxes)
    if (route == CS_A1_TENSOR) return can ? CS_A1_TENSOR : -1;
    const int64_t nT = (N + 255) / 256;
    return can && B * (nT * (nT + 1) / 2) >= TC_MIN_TILES ? CS_A1_TENSOR : CS_A1_FMA;
}

size_t causal_matrix_scratch_bytes(int64_t B, int64_t N, int dim, int geometry, int route)
{
    const int r = resolve_a1_route(B, N, dim, geometry, route);
    return r == CS_A1_TENSOR ? causal_tc_scratch_bytes(B, N, dim, geometry) : 0;
}

// Stream-ordered scratch for callers that pass no workspace: one memory pool per device, owned by the library, which
// keeps what it has allocated (release threshold = never), so that after the first call an allocation is a pointer bump.
int scratch_pool(cudaMemPool_t *out)
{
    static cudaMemPool_t pools[MAX_DEVICES];
    static bool ready[MAX_DEVICES];
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    const int dev = current_device();
    if (!ready[dev]) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        CS_CUDA(cudaMemPoolCreate(&pools[dev], &props));
        uint64_t keep = ~(uint64_t)0;
        CS_CUDA(cudaMemPoolSetAttribute(pools[dev], cudaMemPoolAttrReleaseThreshold, &keep));
        ready[dev] = true;
    }
    *out = pools[dev];
    return CS_OK;
}

// ---- self-check of the tensor route ---------------------------------------------------------------
// The error band of cs_build_tc.cu rests on a model of how the tensor core accumulates (reading A21).  The
// first time CS_A1_AUTO would take the tensor route on a device, the library measures that on the device itself:
// cs_a1_tensor_probe's counters on a seeded causet of 2048 points in 3+1 and in 4+1 dimensions (K = 32 and K = 48 operand
// columns).  If the largest |a - T| reaches a quarter of the margin the device does not behave like the model and AUTO
// keeps the FMA route on it (CS_A1_TENSOR still runs when asked for by name).  Costs ~1 ms and one stream synchronisation, once.
__global__ void k_selfcheck_coords(double *coords, int N, int dim)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    coords[(size_t)i * dim] = -0.9 + 1.8 * (i + 0.5) / N;                    // time: increasing
    uint64_t z = 0x9E3779B97F4A7C15ull * (uint64_t)(i + 1);
    for (int d = 1; d < dim; d++) {                                          // space: SplitMix64 draws in (-0.45, 0.45)
        z += 0x9E3779B97F4A7C15ull;
        uint64_t x = z;
        x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
        x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
        x ^= x >> 31;
        coords[(size_t)i * dim + d] = ((double)(x >> 11) * 0x1p-53 - 0.5) * 0.9;
    }
}

int tensor_route_trusted(cudaStream_t st, bool *trusted)
{
    static std::atomic<int> state[MAX_DEVICES];       // 0 not measured, 1 behaves like the model, 2 does not
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
            const int64_t N = 2048, stride = row_stride_words(N);
            bool ok = true;
            for (int dim = 4; dim <= 5 && ok; dim++) {
                const size_t cb = align_up((size_t)N * dim * 8, 256), mb = align_up((size_t)N * stride * 8, 256);
                const size_t sb = causal_tc_scratch_bytes(1, N, dim, CS_GEOM_MINK_CONE);
                unsigned char *p = nullptr;
                CS_CUDA(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&p), cb + 2 * mb + sb, pool, st));
                double *coords = reinterpret_cast<double *>(p);
                double out[5] = {0, 0, 0, 0, 0};
                rc = [&]() -> int {                       // every exit passes the cudaFreeAsync below
                    k_selfcheck_coords<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(coords, (int)N, dim);
                    CS_LAUNCHED("k_selfcheck_coords");
                    return launch_causal_tc_probe(coords, N, dim, reinterpret_cast<uint64_t *>(p + cb),
                                                  reinterpret_cast<uint64_t *>(p + cb + mb), p + cb + 2 * mb, out, st);   // synchronises
                }();
                cudaFreeAsync(p, st);
                if (rc) return rc;
                ok = out[3] > 0.0 && out[3] < 0.25;
            }
            s0 = ok ? 1 : 2;
            state[dev].store(s0, std::memory_order_release);
        }
    }
    *trusted = s0 == 1;
    return CS_OK;
}

int launch_causal_matrix(const double *coords, int64_t B, int64_t N, int dim, int geometry, int route,
                         uint64_t *bits, uint64_t *bitsT, void *scratch, size_t scratch_bytes, cudaStream_t st)
{
    int r = resolve_a1_route(B, N, dim, geometry, route);
    if (r < 0) return CS_ERR_ARG;
    if (r == CS_A1_TENSOR && route == CS_A1_AUTO) {
        bool trusted = false;
        // a self-check that could not run (say, its pool allocation failed) is no reason to fail the caller: AUTO
        // takes the route that needs no trust, and the check is tried again on the next call
        if (tensor_route_trusted(st, &trusted) != CS_OK) {
            cudaGetLastError();
            trusted = false;
        }
        if (!trusted) r = CS_A1_FMA;
    }
    if (r == CS_A1_FMA) return launch_causal_fma(coords, B, N, dim, geometry, bits, bitsT, st);
    const size_t need = causal_tc_scratch_bytes(B, N, dim, geometry);
    if (scratch) {
        if (scratch_bytes < need || ((uintptr_t)scratch & 255)) return CS_ERR_WORKSPACE;
        return launch_causal_tc(coords, B, N, dim, geometry, bits, bitsT, scratch, st);
    }
    cudaMemPool_t pool;
    int rc = scratch_pool(&pool);
    if (rc) return rc;
    void *p = nullptr;
    CS_CUDA(cudaMallocFromPoolAsync(&p, need, pool, st));
    rc = launch_causal_tc(coords, B, N, dim, geometry, bits, bitsT, p, st);
    cudaError_t e = cudaFreeAsync(p, st);
    if (rc == CS_OK && e != cudaSuccess) return cuda_fail(e, "cudaFreeAsync");
    return rc;
}

// ---- transpose -----------------------------------------------------------------------------
// One warp transposes one 32x32 bit block (transpose32 above); blocks are read as 32-bit halves of the
// uint64 rows.
__global__ void __launch_bounds__(256)
k_transpose_bits(const uint64_t *__restrict__ bits, int64_t N, int64_t stride, uint64_t *__restrict__ bitsT)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t b = blockIdx.z;
    const uint32_t *src = reinterpret_cast<const uint32_t *>(bits + b * N * stride);
    uint32_t *dst = reinterpret_cast<uint32_t *>(bitsT + b * N * stride);
    const int64_t cb = (int64_t)blockIdx.x * 8 + warp;   // 32-column block
    const int64_t rb = blockIdx.y;                       // 32-row block
    const int64_t s32 = stride * 2;
    if (cb >= s32) return;
    const int64_t r = rb * 32 + lane;
    uint32_t x = (r < N) ? src[r * s32 + cb] : 0u;
    x = transpose32(x, lane);
    const int64_t orow = cb * 32 + lane;
    if (orow < N && rb < s32) dst[orow * s32 + rb] = x;
}

__global__ void k_zero_words(uint64_t *p, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0;
}

int launch_transpose_bits(const uint64_t *bits, int64_t B, int64_t N, uint64_t *bitsT, cudaStream_t st)
{
    const int64_t stride = row_stride_words(N);
    if (N == 0) return CS_OK;
    const int64_t s32 = stride * 2;
    const int64_t rblocks = (N + 31) / 32;
    if (rblocks > 65535 || B > 65535) return CS_ERR_ARG;
    if (rblocks < s32) {   // 32-bit words no row block maps to (row padding): clear everything first
        int64_t n = B * N * stride;
        k_zero_words<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(bitsT, n);
        CS_LAUNCHED("k_zero_words");
    }
    dim3 grid((unsigned)((s32 + 7) / 8), (unsigned)rblocks, (unsigned)B);
    k_transpose_bits<<<grid, 256, 0, st>>>(bits, N, stride, bitsT);
    CS_LAUNCHED("k_transpose_bits");
    return CS_OK;
}

// ---- degree vectors -----------------------------------------------------------------------
// out-degree(k) = |J+(k)| = popcount(bits[k]), in-degree(k) = |J-(k)| = popcount(bitsT[k]): the vectors the
// paper's linker accumulates next to the matrix (Alg. 17).  One warp per row.
__global__ void __launch_bounds__(256)
k_degrees(const uint64_t *__restrict__ bits, const uint64_t *__restrict__ bitsT, int64_t N, int64_t stride,
          int64_t *__restrict__ outdeg, int64_t *__restrict__ indeg)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp_global = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t k = warp_global; k < N; k += nwarps) {
        long long o = 0, i = 0;
        for (int64_t w = lane; w < stride; w += 32) {
            o += __popcll(bits[k * stride + w]);
            if (bitsT) i += __popcll(bitsT[k * stride + w]);
        }
#pragma unroll
        for (int s = 16; s >= 1; s >>= 1) {
            o += __shfl_xor_sync(0xffffffffu, o, s);
            i += __shfl_xor_sync(0xffffffffu, i, s);
        }
        if (lane == 0) {
            if (outdeg) outdeg[k] = o;
            if (indeg) indeg[k] = i;
        }
    }
}

int launch_degrees(const uint64_t *bits, const uint64_t *bitsT, int64_t N, int64_t *outdeg, int64_t *indeg, cudaStream_t st)
{
    if (N == 0) return CS_OK;
    const int64_t stride = row_stride_words(N);
    int blocks = sm_count() * 8;
    const int64_t need = (N + 7) / 8;
    if (need < blocks) blocks = (int)need;
    k_degrees<<<blocks, 256, 0, st>>>(bits, bitsT, N, stride, outdeg, indeg);
    CS_LAUNCHED("k_degrees");
    return CS_OK;
}

// ---- relation statistics ------------------------------------------------------------------
// out[0] = R = popcount(bits); out[1] = W_alg = sum_{i -< j} ((j>>6) - (i>>6) + 1)
__global__ void __launch_bounds__(256)
k_relation_stats(const uint64_t *__restrict__ bits, int64_t N, int64_t stride, unsigned long long *out)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp_global = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    unsigned long long R = 0, W = 0;
    for (int64_t i = warp_global; i < N; i += nwarps) {
        const int64_t wi = i >> 6;
        for (int64_t w = wi + lane; w < stride; w += 32) {
            unsigned long long p = __popcll(bits[i * stride + w]);
            R += p;
            W += p * (unsigned long long)(w - wi + 1);
        }
    }
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        R += __shfl_xor_sync(0xffffffffu, R, s);
        W += __shfl_xor_sync(0xffffffffu, W, s);
    }
    if (lane == 0 && (R | W)) {
        atomicAdd(&out[0], R);
        atomicAdd(&out[1], W);
    }
}

int launch_relation_stats(const uint64_t *bits, int64_t N, int64_t *out, cudaStream_t st)
{
    CS_CUDA(cudaMemsetAsync(out, 0, 2 * sizeof(int64_t), st));
    if (N == 0) return CS_OK;
    const int64_t stride = row_stride_words(N);
    int blocks = sm_count() * 8;
    int64_t need = (N + 7) / 8;
    if (need < blocks) blocks = (int)need;
    k_relation_stats<<<blocks, 256, 0, st>>>(bits, N, stride, reinterpret_cast<unsigned long long *>(out));
    CS_LAUNCHED("k_relation_stats");
    return CS_OK;
}

}  // namespace cs
