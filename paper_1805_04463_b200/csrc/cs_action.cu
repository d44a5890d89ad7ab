// cs_action.cu -- stage a3: Benincasa-Dowker action from the interval abundances,
// Eq. 4.10-4.12, l/l_p = 1.  hist[k] = n_{k+1} (Eq. 4.8).
// The bracket is formed exactly in int64; the action is one fp64 multiply.
#include "cs_common.cuh"

namespace cs {

__global__ void k_bd_action(const int64_t *__restrict__ hist, int64_t hist_stride, int64_t B, int64_t kmax,
                            int64_t N, int dim, double *__restrict__ action, int64_t *__restrict__ bracket,
                            int64_t *__restrict__ hist4)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int64_t *h = hist + b * hist_stride;
    const int64_t n1 = (kmax >= 0) ? h[0] : 0;
    const int64_t n2 = (kmax >= 1) ? h[1] : 0;
    const int64_t n3 = (kmax >= 2) ? h[2] : 0;
    const int64_t n4 = (kmax >= 3) ? h[3] : 0;
    int64_t I;
    double S;
    if (dim == 2) {
        I = N - 2 * n1 + 4 * n2 - 2 * n3;
        S = 2.0 * (double)I;
    } else if (dim == 3) {
        // (1/Gamma(5/3)) (pi/(3 sqrt 2))^(2/3), correctly rounded to fp64
        const double c3 = 0x1.d03592b122860p-1;
        I = 8 * N - 8 * n1 + 27 * n2 - 18 * n3;         // 8 x bracket
        S = c3 * ((double)I / 8.0);
    } else {
        const double c4 = 4.0 / 2.449489742783178;       // 4/sqrt(6); sqrt(6) correctly rounded
        I = N - n1 + 9 * n2 - 16 * n3 + 8 * n4;
        S = c4 * (double)I;
    }
    action[b] = S;
    if (bracket) bracket[b] = I;
    if (hist4) {
        hist4[b * 4 + 0] = n1;
        hist4[b * 4 + 1] = n2;
        hist4[b * 4 + 2] = n3;
        hist4[b * 4 + 3] = n4;
    }
}

int launch_bd_action(const int64_t *hist, int64_t hist_stride, int64_t B, int64_t kmax, int64_t N, int dim,
                     double *action, int64_t *bracket, int64_t *hist4, cudaStream_t st)
{
    if (dim < 2 || dim > 4) return CS_ERR_DIM;
    if (B <= 0) return CS_OK;
    k_bd_action<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(hist, hist_stride, B, kmax, N, dim, action, bracket, hist4);
    CS_LAUNCHED("k_bd_action");
    return CS_OK;
}


// ---- smeared (non-local) action, Eq. 4.13-4.18 --------------------------------
//   S_eps = c_d(eps) [ N - a_d eps  sum_k hist[k] f_d(k, eps) ],   a_2 = 2, a_3 = a_4 = 1,
//   f_d(k, eps) = q^k - c1 k eps q^(k-1) + c2 k(k-1) eps^2 q^(k-2) - c3 k(k-1)(k-2) eps^3 q^(k-3),  q = 1 - eps,
// the polynomial form of Eq. 4.16-4.18 (also defined at eps = 1), with (c1, c2, c3) = (2, 1/2, 0),
// (27/8, 9/8, 0), (9, 8, 4/3).  The sum cancels to a small fraction of its terms ("several orders of
// magnitude"), so everything up to the last subtraction is carried in double-double
// (two fp64, error-free transforms with FMA, ~106 bits): q = 1 - eps exactly, q^(k-3) by binary
// powering at the start of a thread's run of k and one multiplication per further k, the bracket as a
// Horner form in q.  One CTA per causet.
namespace {

struct dd { double hi, lo; };

__device__ __forceinline__ dd dd_make(double a) { return dd{a, 0.0}; }
__device__ __forceinline__ dd two_sum(double a, double b)
{
    const double s = a + b, bb = s - a;
    return dd{s, (a - (s - bb)) + (b - bb)};
}
__device__ __forceinline__ dd quick_two_sum(double a, double b)   // |a| >= |b|
{
    const double s = a + b;
    return dd{s, b - (s - a)};
}
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    const dd t = two_sum(a.lo, b.lo);
    s.lo += t.hi;
    s = quick_two_sum(s.hi, s.lo);
    s.lo += t.lo;
    return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    const double p = a.hi * b.hi;
    double e = fma(a.hi, b.hi, -p);
    e = fma(a.hi, b.lo, e);
    e = fma(a.lo, b.hi, e);
    return quick_two_sum(p, e);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b)
{
    const double p = a.hi * b;
    const double e = fma(a.hi, b, -p) + a.lo * b;
    return quick_two_sum(p, e);
}
__device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }

__device__ dd dd_pow(dd q, int64_t n)   // n >= 0
{
    dd r = dd_make(1.0), b = q;
    while (n > 0) {
        if (n & 1) r = dd_mul(r, b);
        b = dd_mul(b, b);
        n >>= 1;
    }
    return r;
}

constexpr int SMEAR_THREADS = 1024;

}  // namespace

__global__ void __launch_bounds__(SMEAR_THREADS)
k_smeared_action(const int64_t *__restrict__ hist, int64_t hist_stride, int64_t kmax, int64_t N, int dim,
                 double eps, double *__restrict__ action)
{
    __shared__ double s_hi[SMEAR_THREADS / 32], s_lo[SMEAR_THREADS / 32];
    const int64_t *h = hist + (int64_t)blockIdx.x * hist_stride;
    const int tid = threadIdx.x;
    const dd q = two_sum(1.0, -eps);                       // exact
    // coefficients as multiples of exactly representable numbers: c1 = n1/8, c2 = n2/8, c3 k(k-1)(k-2) = 4 [k(k-1)(k-2)/3]
    const double n1 = dim == 2 ? 16.0 : dim == 3 ? 27.0 : 72.0;
    const double n2 = dim == 2 ? 4.0 : dim == 3 ? 9.0 : 64.0;
    const dd e1 = dd_make(eps), e2 = dd_mul(e1, e1), e3 = dd_mul(e2, e1);
    const dd q2 = dd_mul(q, q), q3 = dd_mul(q2, q);

    // thread t owns k = t*per .. t*per + per - 1
    const int64_t nk = kmax + 1;
    const int64_t per = (nk + SMEAR_THREADS - 1) / SMEAR_THREADS;
    const int64_t k0 = (int64_t)tid * per, k1 = (k0 + per < nk) ? k0 + per : nk;
    dd sum = dd_make(0.0);
    dd P = dd_make(1.0);                                   // q^(k-3) for k >= 3
    bool have_P = false;
    for (int64_t k = k0; k < k1; k++) {
        const int64_t hk = h[k];
        dd f;
        const double K = (double)k;
        if (k < 3) {   // terms whose falling factorial vanishes are dropped, no negative power is formed
            f = dd_make(1.0);
            if (k == 1) f = dd_add(q, dd_mul_d(e1, -n1 / 8.0));
            if (k == 2) f = dd_add(dd_add(q2, dd_mul_d(dd_mul(e1, q), -2.0 * n1 / 8.0)), dd_mul_d(e2, 2.0 * n2 / 8.0));
        } else {
            if (!have_P) { P = dd_pow(q, k - 3); have_P = true; }
            else P = dd_mul(P, q);
            if (hk == 0) continue;
            // bracket = q^3 - c1 k e q^2 + c2 k(k-1) e^2 q - c3 k(k-1)(k-2) e^3   (all integers below are < 2^53)
            dd br = dd_add(q3, dd_mul_d(dd_mul(e1, q2), -(n1 * K) / 8.0));
            br = dd_add(br, dd_mul_d(dd_mul(e2, q), (n2 * (K * (K - 1.0))) / 8.0));
            if (dim == 4) {
                const double c3k = 4.0 * (double)((k * (k - 1) * (k - 2)) / 3);
                br = dd_add(br, dd_neg(dd_mul_d(e3, c3k)));
            }
            f = dd_mul(P, br);
        }
        if (hk) sum = dd_add(sum, dd_mul_d(f, (double)hk));
    }
    // block reduction in double-double
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        dd o;
        o.hi = __shfl_xor_sync(0xffffffffu, sum.hi, s);
        o.lo = __shfl_xor_sync(0xffffffffu, sum.lo, s);
        sum = dd_add(sum, o);
    }
    if ((tid & 31) == 0) { s_hi[tid >> 5] = sum.hi; s_lo[tid >> 5] = sum.lo; }
    __syncthreads();
    if (tid == 0) {
        dd tot = dd_make(0.0);
        for (int w = 0; w < SMEAR_THREADS / 32; w++) tot = dd_add(tot, dd{s_hi[w], s_lo[w]});
        // N - a_d eps sum, still in double-double; then the prefactor in fp64
        const dd scaled = dd_mul(dd_mul_d(e1, dim == 2 ? 2.0 : 1.0), tot);
        const dd br = dd_add(dd_make((double)N), dd_neg(scaled));
        double c;
        if (dim == 2) c = 2.0 * eps;
        else if (dim == 3) c = 0x1.d03592b122860p-1 * cbrt(eps * eps);   // (1/Gamma(5/3)) (pi/(3 sqrt 2))^(2/3) eps^(2/3)
        else c = 4.0 * sqrt(eps / 6.0);
        action[blockIdx.x] = c * (br.hi + br.lo);
    }
}

int launch_smeared_action(const int64_t *hist, int64_t hist_stride, int64_t B, int64_t kmax, int64_t N, int dim,
                          double eps, double *action, cudaStream_t st)
{
    if (dim < 2 || dim > 4) return CS_ERR_DIM;
    if (!(eps > 0.0 && eps <= 1.0)) return CS_ERR_ARG;
    if (N >= ((int64_t)1 << 17) + 2) return CS_ERR_ARG;   // k(k-1)(k-2) must stay below 2^53
    if (B <= 0) return CS_OK;
    k_smeared_action<<<(unsigned)B, SMEAR_THREADS, 0, st>>>(hist, hist_stride, kmax, N, dim, eps, action);
    CS_LAUNCHED("k_smeared_action");
    return CS_OK;
}

}  // namespace cs
