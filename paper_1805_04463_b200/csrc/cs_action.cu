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

}  // namespace cs
