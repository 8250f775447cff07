/*
 * crmsd_oracle.c -- FP64 CPU oracle for the coordinate RMSD (cRMSD) of protein models.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path (paper_1302_4000_b200/csrc) and is deliberately
 * plain and slow: one pair at a time, in double precision, by the textbook route.
 *
 * What it computes (every citation is /root/reference/PAPER.md:<line>):
 *
 *   cRMSD is DEFINED by eq. 1: sqrt((1/L) sum_i |x_i^A - x_i^B|^2) "after the
 *   optimal superimposition" -- the minimum over proper rotations and translations (Kabsch, ref.
 *   [1]).  The paper's eq. 2 reaches the same number without a
 *   rotation matrix.  The minimum is unique, so the oracle is the plain definition written out:
 *
 *     1. centre both models on their centroids (optimal translation);
 *     2. R_A^2 = (1/L) sum |a_i|^2, R_B^2 likewise (radius of gyration);
 *     3. M = (1/L) sum_i a_i b_i^T  (the 3x3 covariance matrix; normalisation is
 *        reading Q2 of DESIGN.md);
 *     4. singular values s1 >= s2 >= s3 >= 0 of M by one-sided Jacobi (Hestenes) sweeps -- an
 *        SVD, i.e. exactly the route the paper's cubic avoids;
 *     5. S = sign det M (det by cofactor expansion; S = +1 when det >= 0, reading Q4);
 *     6. c^2 = max(0, R_A^2 + R_B^2 - 2 (s1 + s2 + S s3)),  c = sqrt(c^2).
 *
 *   Two more routes are provided so the tests can pin step 4-6 against the paper's own text:
 *     crmsd_pair_eq2   -- eq. 2 literally: eigenvalues of M^T M ("the square of the covariance
 *                         matrix") by a symmetric Jacobi eigen-solver, sqrt, S on the
 *                         smallest (no cubic formula: that is the GPU's route);
 *     crmsd_pair_eq1   -- eq. 1 literally: build the optimal proper rotation from the Jacobi
 *                         factors and sum the residual |a_i - R b_i|^2 atom by atom.
 *
 * Parity pins (tests/test_oracle_pins.py): identity, rigid copy, mirror closed form 2*sqrt(g3),
 * uniform scaling |1-s| R_g, two-atom closed form, planar mirror, symmetry, triangle inequality,
 * bounds, eq.1 == eq.2 == SVD route, brute-force rotation search on tiny inputs, LAPACK SVD on a
 * sample, noise law.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (no -ffast-math).  Inputs are the fp32 arrays the GPU
 * gets, widened to double on load.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- step 1 + 2: centring and R^2 ------------------------------------------------------------ */

/* x[L][3] fp32 -> a[L][3] double centred on the centroid; returns R^2 = (1/L) sum |a_i|^2. */
static double centre_model(const float *x, int L, double *a)
{
    double m[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < L; ++i)
        for (int p = 0; p < 3; ++p) m[p] += (double)x[3 * i + p];
    for (int p = 0; p < 3; ++p) m[p] /= (double)L;
    double r2 = 0.0;
    for (int i = 0; i < L; ++i)
        for (int p = 0; p < 3; ++p) {
            double v = (double)x[3 * i + p] - m[p];
            a[3 * i + p] = v;
            r2 += v * v;
        }
    return r2 / (double)L;
}

/* ---- step 3: covariance ---------------------------------------------------------------------- */

static void covariance(const double *a, const double *b, int L, double M[3][3])
{
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q) M[p][q] = 0.0;
    for (int i = 0; i < L; ++i)
        for (int p = 0; p < 3; ++p)
            for (int q = 0; q < 3; ++q) M[p][q] += a[3 * i + p] * b[3 * i + q];
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q) M[p][q] /= (double)L;
}

static double det3(const double M[3][3])
{
    return M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1])
         - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
         + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
}

/* ---- step 4: one-sided Jacobi SVD of a 3x3 matrix --------------------------------------------- */
/*
 * Hestenes: rotate pairs of COLUMNS of W (initially M) by plane rotations accumulated in V until
 * the columns are mutually orthogonal; then M V = W, the singular values are the column norms and
 * U = W diag(1/s).  Output: s[3] sorted descending, U and V (columns permuted alike) so that
 * M = U diag(s) V^T.  Columns of U belonging to s = 0 are completed to an orthonormal basis.
 */
static void jacobi_svd3(const double M[3][3], double s[3], double U[3][3], double V[3][3])
{
    double W[3][3];
    memcpy(W, M, sizeof W);
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q) V[p][q] = (p == q) ? 1.0 : 0.0;

    for (int sweep = 0; sweep < 60; ++sweep) {
        int rotated = 0;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                double alpha = 0.0, beta = 0.0, gamma = 0.0;
                for (int k = 0; k < 3; ++k) {
                    alpha += W[k][p] * W[k][p];
                    beta += W[k][q] * W[k][q];
                    gamma += W[k][p] * W[k][q];
                }
                if (gamma == 0.0 || fabs(gamma) <= 1e-15 * sqrt(alpha * beta)) continue;
                rotated = 1;
                double zeta = (beta - alpha) / (2.0 * gamma);
                double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                double c = 1.0 / sqrt(1.0 + t * t), sn = c * t;
                for (int k = 0; k < 3; ++k) {
                    double wp = W[k][p], wq = W[k][q];
                    W[k][p] = c * wp - sn * wq;
                    W[k][q] = sn * wp + c * wq;
                    double vp = V[k][p], vq = V[k][q];
                    V[k][p] = c * vp - sn * vq;
                    V[k][q] = sn * vp + c * vq;
                }
            }
        if (!rotated) break;
    }
    double nrm[3];
    int ord[3] = {0, 1, 2};
    for (int q = 0; q < 3; ++q)
        nrm[q] = sqrt(W[0][q] * W[0][q] + W[1][q] * W[1][q] + W[2][q] * W[2][q]);
    for (int i = 0; i < 2; ++i)                     /* sort descending */
        for (int j = 0; j < 2 - i; ++j)
            if (nrm[ord[j]] < nrm[ord[j + 1]]) { int t = ord[j]; ord[j] = ord[j + 1]; ord[j + 1] = t; }
    double Vs[3][3];
    for (int q = 0; q < 3; ++q) {
        s[q] = nrm[ord[q]];
        for (int k = 0; k < 3; ++k) {
            Vs[k][q] = V[k][ord[q]];
            U[k][q] = (s[q] > 0.0) ? W[k][ord[q]] / s[q] : 0.0;
        }
    }
    memcpy(V, Vs, sizeof Vs);
    /* complete U for vanishing singular values (rank-deficient M): Gram-Schmidt on unit vectors */
    for (int q = 0; q < 3; ++q) {
        double n2 = U[0][q] * U[0][q] + U[1][q] * U[1][q] + U[2][q] * U[2][q];
        if (n2 > 0.5) continue;
        double best[3] = {0, 0, 0}, bestn = -1.0;
        for (int e = 0; e < 3; ++e) {
            double v[3] = {0, 0, 0};
            v[e] = 1.0;
            for (int r = 0; r < 3; ++r) {
                if (r == q) continue;
                double nr = U[0][r] * U[0][r] + U[1][r] * U[1][r] + U[2][r] * U[2][r];
                if (nr < 0.5) continue;
                double d = v[0] * U[0][r] + v[1] * U[1][r] + v[2] * U[2][r];
                for (int k = 0; k < 3; ++k) v[k] -= d * U[k][r];
            }
            double vn = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            if (vn > bestn) { bestn = vn; memcpy(best, v, sizeof best); }
        }
        for (int k = 0; k < 3; ++k) U[k][q] = best[k] / bestn;
    }
}

/* ---- steps 4-6 for one pair of CENTRED models ------------------------------------------------ */

/* Returns c^2 (clamped at 0).  The definition route: Jacobi SVD of M. */
static double crmsd2_centred(const double *a, double ra2, const double *b, double rb2, int L)
{
    double M[3][3], s[3], U[3][3], V[3][3];
    covariance(a, b, L, M);
    jacobi_svd3(M, s, U, V);
    double S = (det3(M) >= 0.0) ? 1.0 : -1.0;
    double E = s[0] + s[1] + S * s[2];
    double c2 = ra2 + rb2 - 2.0 * E;
    return c2 > 0.0 ? c2 : 0.0;
}

/* ---- symmetric Jacobi eigen-solver (for the eq. 2 literal route) ----------------------------- */

static void jacobi_eig3(double A[3][3], double lam[3])
{
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = fabs(A[0][1]) + fabs(A[0][2]) + fabs(A[1][2]);
        double dia = fabs(A[0][0]) + fabs(A[1][1]) + fabs(A[2][2]);
        if (off <= 1e-15 * dia || off == 0.0) break;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                if (A[p][q] == 0.0) continue;
                double theta = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double c = 1.0 / sqrt(t * t + 1.0), sn = t * c;
                double R[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
                R[p][p] = c; R[q][q] = c; R[p][q] = sn; R[q][p] = -sn;
                double T[3][3], B[3][3];
                for (int i = 0; i < 3; ++i)          /* T = A R */
                    for (int j = 0; j < 3; ++j) {
                        T[i][j] = 0.0;
                        for (int k = 0; k < 3; ++k) T[i][j] += A[i][k] * R[k][j];
                    }
                for (int i = 0; i < 3; ++i)          /* B = R^T T */
                    for (int j = 0; j < 3; ++j) {
                        B[i][j] = 0.0;
                        for (int k = 0; k < 3; ++k) B[i][j] += R[k][i] * T[k][j];
                    }
                memcpy(A, B, sizeof B);
            }
    }
    lam[0] = A[0][0]; lam[1] = A[1][1]; lam[2] = A[2][2];
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2 - i; ++j)
            if (lam[j] < lam[j + 1]) { double t = lam[j]; lam[j] = lam[j + 1]; lam[j + 1] = t; }
}

/* =============================== exported entry points ======================================= */

/* Steps 1-2 for N models.  centred[N][L][3] (may be NULL), r2[N]. */
void oracle_center(const float *coords, int64_t N, int32_t L, double *centred, double *r2)
{
    #pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        #pragma omp for schedule(static)
        for (int64_t n = 0; n < N; ++n) {
            r2[n] = centre_model(coords + (size_t)n * L * 3, L, a);
            if (centred) memcpy(centred + (size_t)n * L * 3, a, sizeof(double) * 3 * (size_t)L);
        }
        free(a);
    }
}

/* One pair, definition route (steps 1-6).  Returns c; *c2_out = c^2 if not NULL. */
double oracle_crmsd_pair(const float *xa, const float *xb, int32_t L, double *c2_out)
{
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double ra2 = centre_model(xa, L, a), rb2 = centre_model(xb, L, b);
    double c2 = crmsd2_centred(a, ra2, b, rb2, L);
    free(a); free(b);
    if (c2_out) *c2_out = c2;
    return sqrt(c2);
}

/* One pair, eq. 2 literally: eigenvalues of M^T M, descending, sqrt, S on the
 * smallest.  Returns c; writes c^2, the three lambdas and S if the pointers are not NULL. */
double oracle_crmsd_pair_eq2(const float *xa, const float *xb, int32_t L, double *c2_out,
                             double *lambda_out, double *S_out)
{
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double ra2 = centre_model(xa, L, a), rb2 = centre_model(xb, L, b);
    double M[3][3], K[3][3], lam[3];
    covariance(a, b, L, M);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            K[i][j] = 0.0;
            for (int k = 0; k < 3; ++k) K[i][j] += M[k][i] * M[k][j];      /* M^T M */
        }
    jacobi_eig3(K, lam);
    double S = (det3(M) >= 0.0) ? 1.0 : -1.0;
    double E = 0.0;
    for (int k = 0; k < 3; ++k) {
        double l = lam[k] > 0.0 ? lam[k] : 0.0;
        E += (k == 2 ? S : 1.0) * sqrt(l);
        if (lambda_out) lambda_out[k] = lam[k];
    }
    double c2 = ra2 + rb2 - 2.0 * E;
    if (c2 < 0.0) c2 = 0.0;
    free(a); free(b);
    if (c2_out) *c2_out = c2;
    if (S_out) *S_out = S;
    return sqrt(c2);
}

/* One pair, eq. 1 literally: explicit optimal proper rotation R = U D V^T with
 * D = diag(1,1,det(U V^T)), residual summed atom by atom.  Returns c; rot[9] row-major if not NULL. */
double oracle_crmsd_pair_eq1(const float *xa, const float *xb, int32_t L, double *c2_out, double *rot)
{
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    centre_model(xa, L, a);
    centre_model(xb, L, b);
    double M[3][3], s[3], U[3][3], V[3][3], UVt[3][3], R[3][3];
    covariance(a, b, L, M);
    jacobi_svd3(M, s, U, V);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            UVt[i][j] = 0.0;
            for (int k = 0; k < 3; ++k) UVt[i][j] += U[i][k] * V[j][k];
        }
    double d = det3(UVt) >= 0.0 ? 1.0 : -1.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            R[i][j] = U[i][0] * V[j][0] + U[i][1] * V[j][1] + d * U[i][2] * V[j][2];
    double acc = 0.0;
    for (int i = 0; i < L; ++i)
        for (int p = 0; p < 3; ++p) {
            double rb = R[p][0] * b[3 * i] + R[p][1] * b[3 * i + 1] + R[p][2] * b[3 * i + 2];
            double diff = a[3 * i + p] - rb;
            acc += diff * diff;
        }
    double c2 = acc / (double)L;
    free(a); free(b);
    if (c2_out) *c2_out = c2;
    if (rot) memcpy(rot, R, sizeof R);
    return sqrt(c2);
}

/* Singular values of one pair's M, descending, plus det M (for tests). */
void oracle_pair_spectrum(const float *xa, const float *xb, int32_t L, double *s_out, double *det_out,
                          double *M_out)
{
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    centre_model(xa, L, a);
    centre_model(xb, L, b);
    double M[3][3], U[3][3], V[3][3];
    covariance(a, b, L, M);
    jacobi_svd3(M, s_out, U, V);
    if (det_out) *det_out = det3(M);
    if (M_out) memcpy(M_out, M, sizeof M);
    free(a); free(b);
}

/* All-versus-all rows [row_begin, row_end): for each i in the range and every j > i,
 * out[idx] = c(i,j) with idx = packed(i,j) - packed(row_begin,row_begin+1), i.e. the slice of the
 * row-major packed upper triangle (N(N-1)/2 values) that those rows own.
 * c2_out (same indexing) may be NULL.  row range [0,N) gives the whole matrix. */
void oracle_crmsd_rows(const float *coords, int64_t N, int32_t L, int64_t row_begin, int64_t row_end,
                       double *c_out, double *c2_out)
{
    double *cen = (double *)malloc(sizeof(double) * (size_t)N * L * 3);
    double *r2 = (double *)malloc(sizeof(double) * (size_t)N);
    oracle_center(coords, N, L, cen, r2);
    int64_t base = row_begin * (2 * N - row_begin - 1) / 2;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = row_begin; i < row_end; ++i) {
        int64_t off = i * (2 * N - i - 1) / 2 - base;
        const double *a = cen + (size_t)i * L * 3;
        for (int64_t j = i + 1; j < N; ++j) {
            double c2 = crmsd2_centred(a, r2[i], cen + (size_t)j * L * 3, r2[j], L);
            if (c2_out) c2_out[off + (j - i - 1)] = c2;
            c_out[off + (j - i - 1)] = sqrt(c2);
        }
    }
    free(cen); free(r2);
}

/* Listed pairs: c_out[k] = c(pi[k], pj[k]). */
void oracle_crmsd_pairs(const float *coords, int64_t N, int32_t L, const int64_t *pi, const int64_t *pj,
                        int64_t n_pairs, double *c_out, double *c2_out)
{
    (void)N;
    #pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        double *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        #pragma omp for schedule(static)
        for (int64_t k = 0; k < n_pairs; ++k) {
            double ra2 = centre_model(coords + (size_t)pi[k] * L * 3, L, a);
            double rb2 = centre_model(coords + (size_t)pj[k] * L * 3, L, b);
            double c2 = crmsd2_centred(a, ra2, b, rb2, L);
            if (c2_out) c2_out[k] = c2;
            c_out[k] = sqrt(c2);
        }
        free(a); free(b);
    }
}

/* One native against N models. */
void oracle_crmsd_one_vs_all(const float *native, const float *coords, int64_t N, int32_t L,
                             double *c_out, double *c2_out)
{
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    double ra2 = centre_model(native, L, a);
    #pragma omp parallel
    {
        double *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        #pragma omp for schedule(static)
        for (int64_t n = 0; n < N; ++n) {
            double rb2 = centre_model(coords + (size_t)n * L * 3, L, b);
            double c2 = crmsd2_centred(a, ra2, b, rb2, L);
            if (c2_out) c2_out[n] = c2;
            c_out[n] = sqrt(c2);
        }
        free(b);
    }
    free(a);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
