/*
 * causet_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, obviously-correct CPU restatement of the causal-set action
 * path of W. J. Cunningham, "High Performance Algorithms for Quantum Gravity
 * and Cosmology" (arXiv:1805.04463), written from PAPER.md only.  It shares no
 * code with the CUDA path under paper_1805_04463_b200/csrc/ and neither
 * includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.
 *
 * Stages (citations are PAPER.md line numbers):
 *   1. causal matrix:  C[i][j] = (i<j) && pred(x_i, x_j), elements sorted by
 *      time (upper-triangular matrix P).
 *   2. interval abundances:
 *        tier-0  Algorithm 19, literal triple loop
 *        tier-1  Algorithm 20, AND + popcount over the blocks that hold
 *                columns i..j of the symmetrised matrix (PAPER.md:1851-1893,
 *                partial intersection PAPER.md:1066-1068, Fig. 4.2 caption 1768)
 *      hist[k] = #{ i<j related : |A_ij| = k },  i.e. hist[k] = n_{k+1} in the
 *      paper's notation L_m = {i : |A_ij| = m-1} (Eq. 4.8).
 *   3. Benincasa-Dowker action, Eq. 4.10-4.12, l/l_p := 1.
 *   4. (NEXT-1) smeared action, Eq. 4.13-4.18.
 *   5. (NEXT-3) longest chains (Algorithm 11) and the greedy maximal antichain
 *      (Algorithm 13).
 *   6. (NEXT-4) the FLRW relation of Eq. 7.7 as a fourth predicate of stage 1; the flat cone
 *      in 4+1 dimensions (the 4+1 diamond of App. A.1.2); the 3+1 de Sitter slab with
 *      spherical foliation (App. A.1.3) as a fifth predicate.
 *
 * Floating point: every predicate is evaluated in fp64 exactly in the order
 * written below; compile with -ffp-contract=off (no FMA), no -ffast-math.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_chains.py): chain / antichain closed forms, brute-force
 * subset enumeration on N<=64, exhaustive N<=5, sum_k N_k = R,
 * sum_k k N_k = sum_m indeg(m) outdeg(m), inversion-count R and a summed-area
 * table histogram for the 1+1 light-cone diamond, three independent statements
 * of the action coefficients.  "parity unpinned": absolute N_k / action values
 * on random sprinklings (the paper prints none; Fig. 4.5 is an image).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_GEOM_MINK2_LIGHTCONE = 0, ORC_GEOM_MINK_CONE = 1, ORC_GEOM_DS2_SLAB = 2, ORC_GEOM_FLRW_POLAR = 3,
       ORC_GEOM_DS4_SPHERICAL = 4 };

/* 2*pi as the fp64 nearest to the real number (bit pattern 0x401921FB54442D18). */
static const double ORC_TWO_PI = 6.283185307179586476925286766559;

/* ---- stage 1: the relation i -< j between two sprinkled points -------------
 * xi, xj point at `dim` doubles, time coordinate first.
 *  MINK2_LIGHTCONE: light-cone coordinates (u,v), ds^2 = -2 du dv
 *                   (PAPER.md:3717): j in the future of i iff du>0 and dv>0.
 *  MINK_CONE:       (t,x[,y[,z]]): dt >= 0 and dt^2 >= |dx|^2 (timelike or
 *                   null; PAPER.md:1418 with the squared form of Eq. 7.7,
 *                   PAPER.md:3188; readings A1, A2).
 *  DS2_SLAB:        (eta,theta), metric conformal to the cylinder (Eq. 4.19,
 *                   PAPER.md:1949-1951): d_eta >= min(|d_theta|, 2pi-|d_theta|)
 *                   (readings A1, A3).
 *  FLRW_POLAR:      (NEXT-4) conformally flat 3+1 FLRW in conformal time and spherical coordinates,
 *                   Eq. 7.7 as printed, strict:
 *                     r_i^2 + r_j^2 - 2 r_i r_j (cos th_i cos th_j + sin th_i sin th_j cos(ph_i - ph_j)) < (eta_i - eta_j)^2
 *                   A point is (eta, r, cos th, sin th, cos ph, sin ph): the trigonometric values are inputs
 *                   (taken once per point, not once per pair), and cos(ph_i - ph_j) is expanded as
 *                   cos ph_i cos ph_j + sin ph_i sin ph_j, so the predicate is additions and multiplications
 *                   only (reading A17).  j is in the future of i only if eta_j > eta_i.
 *  DS4_SPHERICAL:   (NEXT-4) 3+1 de Sitter, spherical foliation: ds^2 = lambda^2 sec^2(eta) (-d eta^2 + d Omega_3^2)
 *                   (PAPER.md:3845-3847), conformal to R x S^3.  In conformal time "timelike ... intervals
 *                   correspond to d eta^2 > d Sigma^2"; on the unit 3-sphere d Sigma is the
 *                   great-circle angle omega between the two points, cos omega = X_i . X_j with X the unit
 *                   4-vector (cos psi, sin psi cos th, sin psi sin th cos ph, sin psi sin th sin ph).  For
 *                   0 < d eta <= pi (a slab eta in [0, eta0], eta0 < pi/2) and omega in [0, pi] the cosine is
 *                   decreasing, so  d eta > omega  <=>  cos(d eta) < cos omega.  A point is
 *                   (eta, cos eta, sin eta, X0, X1, X2, X3) -- as for FLRW_POLAR the trigonometric values are
 *                   inputs -- and cos(d eta) = cos eta_i cos eta_j + sin eta_i sin eta_j, so the predicate is
 *                   additions and multiplications only, strict, eta_j > eta_i (reading A18).
 *  MINK_CONE dim 5: the same squared form with a fourth spatial coordinate (4+1 diamond).
 */
int orc_relation(const double *xi, const double *xj, int dim, int geom)
{
    if (geom == ORC_GEOM_MINK2_LIGHTCONE) {
        return (xi[0] < xj[0]) && (xi[1] < xj[1]);
    } else if (geom == ORC_GEOM_MINK_CONE) {
        double dt = xj[0] - xi[0];
        double dx = xj[1] - xi[1];
        double s = dx * dx;
        if (dim >= 3) {
            double dy = xj[2] - xi[2];
            s = s + dy * dy;
        }
        if (dim >= 4) {
            double dz = xj[3] - xi[3];
            s = s + dz * dz;
        }
        if (dim >= 5) {
            double dw = xj[4] - xi[4];
            s = s + dw * dw;
        }
        return (dt >= 0.0) && (dt * dt >= s);
    } else if (geom == ORC_GEOM_DS2_SLAB) {
        double deta = xj[0] - xi[0];
        double a = fabs(xj[1] - xi[1]);
        double b = ORC_TWO_PI - a;
        double m = (a < b) ? a : b;
        return deta >= m;
    } else if (geom == ORC_GEOM_FLRW_POLAR) {
        double deta = xj[0] - xi[0];
        double cphi = (xi[4] * xj[4]) + (xi[5] * xj[5]);
        double ang = (xi[2] * xj[2]) + ((xi[3] * xj[3]) * cphi);
        double d2 = ((xi[1] * xi[1]) + (xj[1] * xj[1])) - ((2.0 * (xi[1] * xj[1])) * ang);
        return (deta > 0.0) && (d2 < deta * deta);
    } else if (geom == ORC_GEOM_DS4_SPHERICAL) {
        double deta = xj[0] - xi[0];
        double cd = (xi[1] * xj[1]) + (xi[2] * xj[2]);                                          /* cos(d eta) */
        double co = ((xi[3] * xj[3]) + (xi[4] * xj[4])) + ((xi[5] * xj[5]) + (xi[6] * xj[6]));  /* cos(omega) */
        return (deta > 0.0) && (cd < co);
    }
    return 0;
}

static int orc_geom_ok(int dim, int geom)
{
    if (geom == ORC_GEOM_MINK2_LIGHTCONE) return dim == 2;
    if (geom == ORC_GEOM_MINK_CONE) return dim >= 2 && dim <= 5;
    if (geom == ORC_GEOM_DS2_SLAB) return dim == 2;
    if (geom == ORC_GEOM_FLRW_POLAR) return dim == 6;
    if (geom == ORC_GEOM_DS4_SPHERICAL) return dim == 7;
    return 0;
}

/* Byte matrix C[i*N+j] in {0,1}; only i<j is tested. */
int orc_causal_matrix_bytes(const double *coords, int64_t N, int dim, int geom, uint8_t *C)
{
    if (!orc_geom_ok(dim, geom) || N < 0) return -1;
    memset(C, 0, (size_t)N * (size_t)N);
    for (int64_t i = 0; i < N; i++)
        for (int64_t j = i + 1; j < N; j++)
            C[i * N + j] = (uint8_t)orc_relation(coords + i * dim, coords + j * dim, dim, geom);
    return 0;
}

/* Bit-packed rows (FastBitset layout): row i is
 * `stride` uint64 blocks; element j is bit (j & 63) of block (j >> 6), LSB
 * first; padding bits are zero.  Rows are independent, OpenMP over rows. */
int orc_causal_matrix_bits(const double *coords, int64_t N, int dim, int geom,
                           uint64_t *bits, int64_t stride)
{
    if (!orc_geom_ok(dim, geom) || N < 0 || stride * 64 < N) return -1;
    memset(bits, 0, (size_t)N * (size_t)stride * sizeof(uint64_t));
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; i++)
        for (int64_t j = i + 1; j < N; j++)
            if (orc_relation(coords + i * dim, coords + j * dim, dim, geom))
                bits[i * stride + (j >> 6)] |= (uint64_t)1 << (j & 63);
    return 0;
}

/* Transposed copy: bitsT[j] holds the past of j (bit i set iff i -< j). */
void orc_transpose_bits(const uint64_t *bits, int64_t N, int64_t stride, uint64_t *bitsT)
{
    memset(bitsT, 0, (size_t)N * (size_t)stride * sizeof(uint64_t));
    for (int64_t i = 0; i < N; i++)
        for (int64_t b = 0; b < stride; b++) {
            uint64_t w = bits[i * stride + b];
            while (w) {                                   /* visit the set bits of the block */
                int64_t j = b * 64 + __builtin_ctzll(w);
                w &= w - 1;
                if (j < N) bitsT[j * stride + (i >> 6)] |= (uint64_t)1 << (i & 63);
            }
        }
}

/* out-degree (row sums) and in-degree (column sums) of the relation. */
void orc_degrees(const uint64_t *bits, int64_t N, int64_t stride, int64_t *outdeg, int64_t *indeg)
{
    for (int64_t i = 0; i < N; i++) { outdeg[i] = 0; indeg[i] = 0; }
    for (int64_t i = 0; i < N; i++)
        for (int64_t b = 0; b < stride; b++) {
            uint64_t w = bits[i * stride + b];
            while (w) {
                int64_t j = b * 64 + __builtin_ctzll(w);
                w &= w - 1;
                if (j < N) { outdeg[i]++; indeg[j]++; }
            }
        }
}

void orc_pack_bytes(const uint8_t *C, int64_t N, uint64_t *bits, int64_t stride)
{
    memset(bits, 0, (size_t)N * (size_t)stride * sizeof(uint64_t));
    for (int64_t i = 0; i < N; i++)
        for (int64_t j = 0; j < N; j++)
            if (C[i * N + j]) bits[i * stride + (j >> 6)] |= (uint64_t)1 << (j & 63);
}

void orc_unpack_bits(const uint64_t *bits, int64_t N, int64_t stride, uint8_t *C)
{
    for (int64_t i = 0; i < N; i++)
        for (int64_t j = 0; j < N; j++)
            C[i * N + j] = (uint8_t)((bits[i * stride + (j >> 6)] >> (j & 63)) & 1);
}

/* ---- stage 2, tier-0: Algorithm 19, literally ---------
 * for i, for j>i, skip unless i -< j; x = #{k in (i,j): i -< k and k -< j};
 * n[x+1]++.  (The listing omits the per-pair reset x <- 0; A4.)
 * hist has N-1 entries, k = 0..N-2 ("largest possible ... N-2 elements",
 * PAPER.md:1839).  hist[k] = n[k+1]. */
void orc_interval_hist_alg19(const uint8_t *C, int64_t N, int64_t *hist)
{
    for (int64_t k = 0; k < N - 1; k++) hist[k] = 0;
    for (int64_t i = 0; i < N - 1; i++) {
        for (int64_t j = i + 1; j < N; j++) {
            if (!C[i * N + j]) continue;
            int64_t x = 0;
            for (int64_t k = i + 1; k < j; k++)
                if (C[i * N + k] && C[k * N + j]) x++;
            hist[x]++;
        }
    }
}

/* ---- stage 2, tier-1: Algorithm 20 --------------------
 * Works on the symmetrised matrix A = P + P^T kept as
 * uint64 rows.  For every related pair (i,j), i<j:
 *     m = A[i].PARTIAL_VECPROD(A[j], offset i, length j-i+1)     (line 9)
 * = popcount of (A[i] AND A[j]) restricted to bit positions i..j, everything
 * outside zeroed.  Bits i and j themselves are 0
 * (irreflexive), so the closed range counts exactly the open interval.
 * Restricted to rows i = row_begin, row_begin+row_step, ... < row_end.
 * Per-thread histograms, then the reduction of lines 12-14.  *word_ops
 * accumulates the number of 64-bit blocks touched, sum over related pairs of
 * (j>>6)-(i>>6)+1; *loop_seconds is the wall time of the pair loop alone (the
 * paper's linker already delivers the symmetrised matrix).
 */
static uint64_t orc_mask_from(int b) { return ~(uint64_t)0 << b; }              /* bits b..63 */
static uint64_t orc_mask_upto(int b) { return ~(uint64_t)0 >> (63 - b); }       /* bits 0..b  */

int orc_interval_hist_alg20(const uint64_t *bits, int64_t N, int64_t stride,
                            int64_t row_begin, int64_t row_end, int64_t row_step,
                            int64_t *hist, int64_t *word_ops, double *loop_seconds, int nthreads)
{
    if (N < 0 || stride * 64 < N) return -1;
    int64_t nh = N > 1 ? N - 1 : 0;
    for (int64_t k = 0; k < nh; k++) hist[k] = 0;
    if (word_ops) *word_ops = 0;
    if (N < 2) return 0;
    if (row_begin < 0) row_begin = 0;
    if (row_end > N) row_end = N;
    if (row_step < 1) row_step = 1;
    if (loop_seconds) *loop_seconds = 0.0;

    /* A = P + P^T */
    uint64_t *A = (uint64_t *)malloc((size_t)N * (size_t)stride * sizeof(uint64_t));
    if (!A) return -2;
    orc_transpose_bits(bits, N, stride, A);
    for (int64_t w = 0; w < N * stride; w++) A[w] |= bits[w];

#ifdef _OPENMP
    int T = nthreads > 0 ? nthreads : omp_get_max_threads();
#else
    int T = 1;
    (void)nthreads;
#endif
    int64_t *n = (int64_t *)calloc((size_t)T * (size_t)nh, sizeof(int64_t));
    int64_t *wops = (int64_t *)calloc((size_t)T, sizeof(int64_t));
    if (!n || !wops) { free(A); free(n); free(wops); return -2; }

#ifdef _OPENMP
    double t0 = omp_get_wtime();
#endif
#pragma omp parallel for schedule(dynamic, 1) num_threads(T)
    for (int64_t i = row_begin; i < row_end; i += row_step) {
#ifdef _OPENMP
        int t = omp_get_thread_num();
#else
        int t = 0;
#endif
        const uint64_t *Ai = A + i * stride;
        for (int64_t j = i + 1; j < N; j++) {
            if (!((Ai[j >> 6] >> (j & 63)) & 1)) continue;      /* i not-< j */
            const uint64_t *Aj = A + j * stride;
            int64_t x = i >> 6, y = j >> 6;
            int64_t m = 0;
            if (x == y) {
                uint64_t w = Ai[x] & Aj[x] & orc_mask_from((int)(i & 63)) & orc_mask_upto((int)(j & 63));
                m = __builtin_popcountll(w);
            } else {
                m += __builtin_popcountll(Ai[x] & Aj[x] & orc_mask_from((int)(i & 63)));
                for (int64_t b = x + 1; b < y; b++) m += __builtin_popcountll(Ai[b] & Aj[b]);
                m += __builtin_popcountll(Ai[y] & Aj[y] & orc_mask_upto((int)(j & 63)));
            }
            n[(int64_t)t * nh + m]++;
            wops[t] += y - x + 1;
        }
    }
#ifdef _OPENMP
    if (loop_seconds) *loop_seconds = omp_get_wtime() - t0;
#endif
    for (int t = 0; t < T; t++) {
        for (int64_t m = 0; m < nh; m++) hist[m] += n[(int64_t)t * nh + m];
        if (word_ops) *word_ops += wops[t];
    }
    free(A); free(n); free(wops);
    return T;
}

/* Number of relations R = popcount(bits) and the Alg. 20 block count
 * W_alg = sum_{i -< j} ((j>>6) - (i>>6) + 1), from the bits alone. */
void orc_count_relations(const uint64_t *bits, int64_t N, int64_t stride,
                         int64_t *n_relations, int64_t *word_ops)
{
    int64_t R = 0, W = 0;
    for (int64_t i = 0; i < N; i++)
        for (int64_t j = i + 1; j < N; j++)
            if ((bits[i * stride + (j >> 6)] >> (j & 63)) & 1) {
                R++;
                W += (j >> 6) - (i >> 6) + 1;
            }
    if (n_relations) *n_relations = R;
    if (word_ops) *word_ops = W;
}

/* ---- stage 3: Benincasa-Dowker action, Eq. 4.10-4.12 --
 * n_m = hist[m-1]; entries beyond nhist are 0 (N too small).  l/l_p := 1.
 *   d=2: S = 2 (N - 2 n1 + 4 n2 - 2 n3)
 *   d=3: S = (1/Gamma(5/3)) (pi/(3 sqrt 2))^(2/3) (N - n1 + (27/8) n2 - (9/4) n3)
 *   d=4: S = (4/sqrt 6) (N - n1 + 9 n2 - 16 n3 + 8 n4)
 * The bracket is returned exactly: as int64 for d=2,4 and as an int64 count
 * of eighths (8 x bracket) for d=3, through *bracket_num.
 */
double orc_bd_action(const int64_t *hist, int64_t nhist, int64_t N, int dim, int64_t *bracket_num)
{
    int64_t n1 = nhist > 0 ? hist[0] : 0;
    int64_t n2 = nhist > 1 ? hist[1] : 0;
    int64_t n3 = nhist > 2 ? hist[2] : 0;
    int64_t n4 = nhist > 3 ? hist[3] : 0;
    if (dim == 2) {
        int64_t I = N - 2 * n1 + 4 * n2 - 2 * n3;
        if (bracket_num) *bracket_num = I;
        return 2.0 * (double)I;
    } else if (dim == 3) {
        int64_t I8 = 8 * N - 8 * n1 + 27 * n2 - 18 * n3;
        if (bracket_num) *bracket_num = I8;
        double c3 = (1.0 / tgamma(5.0 / 3.0)) * pow(M_PI / (3.0 * sqrt(2.0)), 2.0 / 3.0);
        return c3 * ((double)I8 / 8.0);
    } else if (dim == 4) {
        int64_t I = N - n1 + 9 * n2 - 16 * n3 + 8 * n4;
        if (bracket_num) *bracket_num = I;
        return (4.0 / sqrt(6.0)) * (double)I;
    }
    if (bracket_num) *bracket_num = 0;
    return NAN;
}

/* ---- smearing functions, Eq. 4.16-4.18 ---------------
 * f_d(m, eps), written in the polynomial form obtained by multiplying the
 * (1-eps)^m prefactor into the bracket, which is also defined at eps = 1
 * (0^0 := 1):
 *   f2 = (1-e)^m - 2 m e (1-e)^(m-1) + [m(m-1)/2] e^2 (1-e)^(m-2)
 *   f3 = (1-e)^m - (27/8) m e (1-e)^(m-1) + (9/8) m(m-1) e^2 (1-e)^(m-2)
 *   f4 = (1-e)^m - 9 m e (1-e)^(m-1) + 8 m(m-1) e^2 (1-e)^(m-2)
 *        - (4/3) m(m-1)(m-2) e^3 (1-e)^(m-3)
 * Terms whose falling factorial vanishes are dropped before the power is
 * formed, so no negative exponent is ever evaluated.
 */
static long double orc_powl_nonneg(long double b, int64_t e)
{
    if (e == 0) return 1.0L;
    return powl(b, (long double)e);
}

static long double orc_smear_fl(int dim, int64_t m, double eps)
{
    long double e = eps, q = 1.0L - e, M = (long double)m;
    long double f = orc_powl_nonneg(q, m);
    if (dim == 2) {
        if (m >= 1) f -= 2.0L * M * e * orc_powl_nonneg(q, m - 1);
        if (m >= 2) f += 0.5L * M * (M - 1) * e * e * orc_powl_nonneg(q, m - 2);
    } else if (dim == 3) {
        if (m >= 1) f -= (27.0L / 8.0L) * M * e * orc_powl_nonneg(q, m - 1);
        if (m >= 2) f += (9.0L / 8.0L) * M * (M - 1) * e * e * orc_powl_nonneg(q, m - 2);
    } else if (dim == 4) {
        if (m >= 1) f -= 9.0L * M * e * orc_powl_nonneg(q, m - 1);
        if (m >= 2) f += 8.0L * M * (M - 1) * e * e * orc_powl_nonneg(q, m - 2);
        if (m >= 3) f -= (4.0L / 3.0L) * M * (M - 1) * (M - 2) * e * e * e * orc_powl_nonneg(q, m - 3);
    } else {
        return (long double)NAN;
    }
    return f;
}

double orc_smear_f(int dim, int64_t m, double eps) { return (double)orc_smear_fl(dim, m, eps); }

/* Smeared action, Eq. 4.13-4.15; sum over m = 1..N-1 of
 * n_m f_d(m-1, eps) = sum_k hist[k] f_d(k, eps); long double accumulation. */
double orc_smeared_action(const int64_t *hist, int64_t nhist, int64_t N, int dim, double eps)
{
    long double sum = 0.0L;
    for (int64_t k = 0; k < nhist; k++)
        if (hist[k]) sum += (long double)hist[k] * orc_smear_fl(dim, k, eps);   /* f_d kept in long double */
    long double e = eps;
    if (dim == 2) return (double)(2.0L * e * ((long double)N - 2.0L * e * sum));
    if (dim == 3) {
        long double c = (1.0L / tgammal(5.0L / 3.0L)) * powl(M_PIl * e / (3.0L * sqrtl(2.0L)), 2.0L / 3.0L);
        return (double)(c * ((long double)N - e * sum));
    }
    if (dim == 4) return (double)(4.0L * sqrtl(e / 6.0L) * ((long double)N - e * sum));
    return NAN;
}

/* ---- NEXT-3: chains and antichains -------------------------------------
 * All three work on the byte matrix C[i*N + j] = (i -< j) of stage 1 (tier-0 style: plain loops).
 *
 * orc_chain_pair: Algorithm 11 literally (text 1326, 1353): for i -< j the
 * recursion moves through the Alexandroff set A_ij = J+(i) & J-(j), L[k] memoises the distance from
 * k to j, unvisited entries are -1.  With l starting at 0 the procedure returns
 * l + 1 = the number of LINKS of the longest chain from i to j (1 if A_ij is empty), i.e. the number
 * of elements of that chain minus one.  Returns 0 if i is not related to j.  (The listing's recursive
 * call passes "A_ki"; the set being scanned must be A_kj, the one formed on the line before it.)
 */
static int64_t orc_chain_rec(const uint8_t *C, int64_t N, int64_t *L, int64_t i, int64_t j)
{
    int64_t l = 0;
    for (int64_t k = i + 1; k < j; k++) {
        if (!(C[i * N + k] && C[k * N + j])) continue;          /* k in A_ij */
        int64_t kappa;
        if (L[k] == -1) {
            int nonempty = 0;
            for (int64_t m = k + 1; m < j && !nonempty; m++) nonempty = C[k * N + m] && C[m * N + j];
            if (nonempty) kappa = orc_chain_rec(C, N, L, k, j);
            else kappa = 1;
            L[k] = kappa;
        } else {
            kappa = L[k];
        }
        if (kappa > l) l = kappa;
    }
    return l + 1;
}

int64_t orc_chain_pair(const uint8_t *C, int64_t N, int64_t i, int64_t j)
{
    if (i < 0 || j >= N || i >= j || !C[i * N + j]) return 0;
    int64_t *L = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    for (int64_t k = 0; k < N; k++) L[k] = -1;
    int64_t r = orc_chain_rec(C, N, L, i, j);
    free(L);
    return r;
}

/* orc_chain_heights: the definition the recursion reaches, written out for every element at once.
 * height[k] = number of elements of the longest chain that ends at k; with source >= 0 only chains
 * that start at `source` count (height[source] = 1, 0 for elements outside J+(source)).  Elements
 * are in time order, so predecessors come first.  Returns the largest height (0 for N = 0). */
int64_t orc_chain_heights(const uint8_t *C, int64_t N, int64_t source, int32_t *height)
{
    int64_t best = 0;
    for (int64_t j = 0; j < N; j++) {
        int32_t h;
        if (source < 0) {
            h = 1;
            for (int64_t i = 0; i < j; i++)
                if (C[i * N + j] && height[i] + 1 > h) h = height[i] + 1;
        } else if (j == source) {
            h = 1;
        } else if (j < source || !C[source * N + j]) {
            h = 0;
        } else {
            h = 2;                                              /* source -< j */
            for (int64_t i = source + 1; i < j; i++)
                if (height[i] > 0 && C[i * N + j] && height[i] + 1 > h) h = height[i] + 1;
        }
        height[j] = h;
        if (h > best) best = h;
    }
    return best;
}

/* orc_greedy_antichain: Algorithm 13 literally (text 1355-1359).  J(j) = J+(j) | J-(j).
 * Candidates Xi = P \ J(seed) \ {seed}, A = {seed} | Xi; while Xi is not empty: for j in Xi in index
 * order c = |A \ J(j)|, keep the FIRST j with the largest c (the listing's strict "c > sigma"), then
 * A = A \ J(k), Xi = Xi \ (J(k) | {k}).  member[] gets 0/1; returns |A|. */
int64_t orc_greedy_antichain(const uint8_t *C, int64_t N, int64_t seed, uint8_t *member)
{
    if (N <= 0 || seed < 0 || seed >= N) return 0;
    uint8_t *xi = (uint8_t *)calloc((size_t)N, 1);
    int64_t nxi = 0;
#define ORC_REL(a, b) (C[(a) * N + (b)] || C[(b) * N + (a)])
    for (int64_t j = 0; j < N; j++) {
        xi[j] = (j != seed) && !ORC_REL(seed, j);
        member[j] = (j == seed) || xi[j];
        nxi += xi[j];
    }
    while (nxi > 0) {
        int64_t sigma = 0, k = -1;
        for (int64_t j = 0; j < N; j++) {
            if (!xi[j]) continue;
            int64_t c = 0;
            for (int64_t a = 0; a < N; a++) c += member[a] && !ORC_REL(j, a);
            if (c > sigma) { sigma = c; k = j; }
        }
        /* c >= 1 always (j itself is in A and not in J(j)), so k is set */
        for (int64_t a = 0; a < N; a++) {
            if (ORC_REL(k, a)) {
                member[a] = 0;
                if (xi[a]) { xi[a] = 0; nxi--; }
            }
        }
        xi[k] = 0;
        nxi--;
    }
#undef ORC_REL
    free(xi);
    int64_t size = 0;
    for (int64_t a = 0; a < N; a++) size += member[a];
    return size;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
