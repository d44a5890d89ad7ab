// cs_predicates.cuh -- the relation predicates of include/causalset.h in fp64 (Pred) and the per-point data of the
// exact single-precision prefilter for predicates that are the sign of a bilinear form (Fast); shared by the two a1
// kernels (cs_build.cu: FMA pipes, cs_build_tc.cu: tensor cores).
#pragma once
#include "cs_common.cuh"

namespace cs {

template <int GEOM, int DIM>
struct Pred;

template <>
struct Pred<CS_GEOM_MINK2_LIGHTCONE, 2> {
    __device__ static __forceinline__ bool rel(const double *xi, const double *xj)
    {
        return (xi[0] < xj[0]) && (xi[1] < xj[1]);
    }
};

template <int DIM>
struct Pred<CS_GEOM_MINK_CONE, DIM> {
    __device__ static __forceinline__ bool rel(const double *xi, const double *xj)
    {
        double dt = __dsub_rn(xj[0], xi[0]);
        double dx = __dsub_rn(xj[1], xi[1]);
        double s = __dmul_rn(dx, dx);
        if (DIM >= 3) {
            double dy = __dsub_rn(xj[2], xi[2]);
            s = __dadd_rn(s, __dmul_rn(dy, dy));
        }
        if (DIM >= 4) {
            double dz = __dsub_rn(xj[3], xi[3]);
            s = __dadd_rn(s, __dmul_rn(dz, dz));
        }
        if (DIM >= 5) {
            double dw = __dsub_rn(xj[4], xi[4]);
            s = __dadd_rn(s, __dmul_rn(dw, dw));
        }
        return (dt >= 0.0) && (__dmul_rn(dt, dt) >= s);
    }
};

template <>
struct Pred<CS_GEOM_DS2_SLAB, 2> {
    __device__ static __forceinline__ bool rel(const double *xi, const double *xj)
    {
        const double two_pi = __longlong_as_double(0x401921FB54442D18LL);
        double deta = __dsub_rn(xj[0], xi[0]);
        double a = fabs(__dsub_rn(xj[1], xi[1]));
        double b = __dsub_rn(two_pi, a);
        double m = (a < b) ? a : b;
        return deta >= m;
    }
};

template <>
struct Pred<CS_GEOM_FLRW_POLAR, 6> {
    __device__ static __forceinline__ bool rel(const double *xi, const double *xj)
    {
        const double deta = __dsub_rn(xj[0], xi[0]);
        const double cphi = __dadd_rn(__dmul_rn(xi[4], xj[4]), __dmul_rn(xi[5], xj[5]));
        const double ang = __dadd_rn(__dmul_rn(xi[2], xj[2]), __dmul_rn(__dmul_rn(xi[3], xj[3]), cphi));
        const double d2 = __dsub_rn(__dadd_rn(__dmul_rn(xi[1], xi[1]), __dmul_rn(xj[1], xj[1])),
                                    __dmul_rn(__dmul_rn(2.0, __dmul_rn(xi[1], xj[1])), ang));
        return (deta > 0.0) && (d2 < __dmul_rn(deta, deta));
    }
};

template <>
struct Pred<CS_GEOM_DS4_SPHERICAL, 7> {
    __device__ static __forceinline__ bool rel(const double *xi, const double *xj)
    {
        const double deta = __dsub_rn(xj[0], xi[0]);
        const double cd = __dadd_rn(__dmul_rn(xi[1], xj[1]), __dmul_rn(xi[2], xj[2]));
        const double co = __dadd_rn(__dadd_rn(__dmul_rn(xi[3], xj[3]), __dmul_rn(xi[4], xj[4])),
                                    __dadd_rn(__dmul_rn(xi[5], xj[5]), __dmul_rn(xi[6], xj[6])));
        return (deta > 0.0) && (cd < co);
    }
};

// ---- exact single-precision prefilter (flat cone) ----------------------------------------------
// With h = (t^2 - |x|^2) / 2 the sign of the interval is the sign of
//     T = ((t_j - t_i)^2 - |x_j - x_i|^2) / 2 = h_i + h_j - t_i t_j + x_i . x_j ,
// four FFMA and one FADD per pair in fp32 instead of twelve fp64-pipe instructions.  The fp32 value a
// differs from T by at most 34 u C^2 (u = 2^-24, C = largest |coordinate| of the tile: 8 input
// roundings <= 8.04 u C^2, two roundings of h <= 3 u C^2, five result roundings of partial sums
// bounded by 2.5, 3.5, 4.5, 5.5 and 7 C^2), so with m = 64 u C^2
//     a >  m  =>  T >  30 u C^2  : related     (the fp64 expression errs by < 2^-46 C^2, and dt >= 0
//     a < -m  =>  T < -30 u C^2  : unrelated    holds for the whole tile, checked below)
// and anything else -- including NaN -- is re-evaluated with the fp64 expression of the header for
// the whole 32 x 32 block.  The output is therefore bit-identical to the plain fp64 evaluation.
// The tile takes this path only if the header's dt >= 0 holds for every pair it keeps (off the
// diagonal: max t_i <= min t_j; diagonal tile: its points are in time order -- always the case for
// time-sorted input) and 2^-40 <= C <= 2^40 (no overflow or underflow in the fp32 products).
//
// de Sitter slab: the same scheme on D = (eta_j - eta_i) - min(|dtheta|, 2pi - |dtheta|), five fp32 operations.
// With C = max(|eta|, |theta|, 2pi) over the tile: the two differences are each off by <= 4 u C (two input
// roundings and the subtraction), b = 2pi - a by <= 8 u C, the minimum by no more, d = deta - m by
// <= 17 u C; margin m = 32 u C.  d > m => D > 15 u C => the fp64 expression (errors ~2^-50 C) says related,
// d < -m => unrelated, else fp64.  No time-order condition: the header's expression has none.
//
// The same scheme covers every predicate that is the sign of a bilinear form  T = sum_c P_c(i) F_c(j) + h_i + h_j :
//   flat cone, dim 2..5      P = (-t, x, ..), F = (t, x, ..), h = (t^2 - |x|^2) / 2
//   FLRW, Eq. 7.7            the flat cone of the Cartesian conformal coordinates (eta, r st cp, r st sp, r ct), formed
//                            per point in fp64.  The header's law-of-cosines value differs from |x_i - x_j|^2 by
//                            r^2 (1 - (ct^2 + st^2 (cp^2 + sp^2))) per point, so a tile takes the fast path only if every
//                            point has ct^2 + st^2 and cp^2 + sp^2 within 2^-30 of 1 (<= 2^-28 C^2 in all, against a
//                            margin of 2^-18 C^2); anything else falls back to the header's fp64 expression.
//   3+1 de Sitter, spherical P = (-cos eta, -sin eta, X0..X3), F = (cos eta, sin eta, X0..X3), no h:
//                            T = cos(omega) - cos(d eta); 12 input roundings + partial sums 1..6 C^2 <= 33 u C^2.
//                            Unit inputs and finite times only, tiles strictly ordered in time (Fast<DS4_SPHERICAL>).
// With NP products the bound is (2.01 NP + (NP - 1) + sum of the partial sums) u C^2: 34 (NP = 4), 48 (NP = 5), so the
// margin is 64 u C^2 up to four products (and for the h-free six of de Sitter) and 96 u C^2 for five.
// The first NNEG components are stored negated for the past point.  convert() returns false for a point that may not
// use the prefilter.
template <int GEOM, int DIM>
struct Fast {
    static constexpr bool ok = false, H = false, STRICT = false;
    static constexpr int NP = 1, NNEG = 0, MARGIN = 64;
    __device__ static __forceinline__ bool convert(const double *, float *, float &) { return false; }
};
template <int DIM>
struct Fast<CS_GEOM_MINK_CONE, DIM> {
    static constexpr bool ok = true, H = true, STRICT = false;
    static constexpr int NP = DIM, NNEG = 1, MARGIN = DIM <= 4 ? 64 : 96;
    __device__ static __forceinline__ bool convert(const double *x, float *v, float &h)
    {
        double sq = 0.0;
#pragma unroll
        for (int d = 0; d < DIM; d++) {
            v[d] = (float)x[d];
            if (d > 0) sq += x[d] * x[d];
        }
        h = (float)(0.5 * (x[0] * x[0] - sq));
        return true;
    }
};
template <>
struct Fast<CS_GEOM_DS2_SLAB, 2> {      // not a bilinear form: its own five-operation expression (above)
    static constexpr bool ok = true, H = false, STRICT = false;
    static constexpr int NP = 2, NNEG = 0, MARGIN = 32;
    __device__ static __forceinline__ bool convert(const double *x, float *v, float &h)
    {
        v[0] = (float)x[0];
        v[1] = (float)x[1];
        h = 0.f;
        return true;
    }
};
template <>
struct Fast<CS_GEOM_DS4_SPHERICAL, 7> {
    // The time coordinate is not part of T (only its cosine and sine columns are), so the header's "eta_j - eta_i > 0"
    // must come from the tile test alone: STRICT asks the callers for max eta_i < min eta_j (and strictly increasing
    // times inside a diagonal tile) instead of <=, and a point whose eta is NaN or infinite -- the header's difference is
    // then NaN for some partner, "unrelated" whatever the other columns say -- does not take the prefilter.
    static constexpr bool ok = true, H = false, STRICT = true;
    static constexpr int NP = 6, NNEG = 2, MARGIN = 64;
    __device__ static __forceinline__ bool convert(const double *x, float *v, float &h)
    {
#pragma unroll
        for (int c = 0; c < 6; c++) v[c] = (float)x[1 + c];
        h = 0.f;
        // inputs that are not unit vectors do not take the prefilter
        const double n1 = x[1] * x[1] + x[2] * x[2] - 1.0;
        const double n2 = (x[3] * x[3] + x[4] * x[4]) + (x[5] * x[5] + x[6] * x[6]) - 1.0;
        return isfinite(x[0]) && fabs(n1) <= 0x1p-30 && fabs(n2) <= 0x1p-30;      // false for NaN
    }
};
template <>
struct Fast<CS_GEOM_FLRW_POLAR, 6> {
    static constexpr bool ok = true, H = true, STRICT = false;
    static constexpr int NP = 4, NNEG = 1, MARGIN = 64;
    __device__ static __forceinline__ bool convert(const double *x, float *v, float &h)
    {
        const double rs = x[1] * x[3];
        const double cx = rs * x[4], cy = rs * x[5], cz = x[1] * x[2];
        v[0] = (float)x[0];
        v[1] = (float)cx;
        v[2] = (float)cy;
        v[3] = (float)cz;
        h = (float)(0.5 * (x[0] * x[0] - (cx * cx + cy * cy + cz * cz)));
        const double n1 = x[2] * x[2] + x[3] * x[3] - 1.0, n2 = x[4] * x[4] + x[5] * x[5] - 1.0;
        return fabs(n1) <= 0x1p-30 && fabs(n2) <= 0x1p-30;      // false for NaN
    }
};

// 32 x 32 bit block held one word per lane (lane = column, bit = row) -> one word per lane
// (lane = row, bit = column): the 5-step butterfly.  Step t exchanges with lane ^ s (s = 16 >> t) and keeps
// x & keep | rot(partner) & ~keep, where the partner word is shifted right by s in the lanes with bit s set
// and left by s in the others; a rotation does both, the bits that wrap around land where ~keep is 0.
// keep[t] and rot[t] depend on the lane only (TransposeLane, set up once per kernel).
struct TransposeLane {
    uint32_t keep[5], rot[5];
    __device__ __forceinline__ explicit TransposeLane(int lane)
    {
        const uint32_t mlo[5] = {0x0000FFFFu, 0x00FF00FFu, 0x0F0F0F0Fu, 0x33333333u, 0x55555555u};
#pragma unroll
        for (int t = 0; t < 5; t++) {
            const int s = 16 >> t;
            keep[t] = (lane & s) ? ~mlo[t] : mlo[t];
            rot[t] = (lane & s) ? 32 - s : s;           // rotate left by 32 - s = shift right by s
        }
    }
    __device__ __forceinline__ uint32_t operator()(uint32_t x) const
    {
#pragma unroll
        for (int t = 0; t < 5; t++) {
            const uint32_t o = __shfl_xor_sync(0xffffffffu, x, 16 >> t);
            const uint32_t r = __funnelshift_l(o, o, rot[t]);
            x = (x & keep[t]) | (r & ~keep[t]);
        }
        return x;
    }
};

__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane) { return TransposeLane(lane)(x); }

// min(u, |a|, |b|), NaN if any operand is NaN (one FMNMX3.NAN)
__device__ __forceinline__ float min3_abs_nan(float u, uint32_t a, uint32_t b)
{
    float d;
    asm("{\n"
        ".reg .f32 x, y;\n"
        "abs.f32 x, %2;\n"
        "abs.f32 y, %3;\n"
        "min.NaN.f32 %0, %1, x, y;\n"
        "}\n" : "=f"(d) : "f"(u), "f"(__uint_as_float(a)), "f"(__uint_as_float(b)));
    return d;
}

}  // namespace cs
