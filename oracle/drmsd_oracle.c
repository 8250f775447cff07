/*
 * drmsd_oracle.c -- FP64 CPU oracle for the distance RMSD (dRMSD) of protein models.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as crmsd_oracle.c: only tests/, smoke() and bench.py's CPU
 * legs may build, load or call it; no code shared with paper_1302_4000_b200/csrc).
 *
 * What it computes: the paper's eq. 5 written out literally,
 *
 *     dRMSD(A,B) = sqrt( 2/(L(L-1)) * sum_{i<j} (d_ij^A - d_ij^B)^2 ),   d_ij = |x_i - x_j|,
 *
 * with the paper's "N" read as the number of atoms L (reading Q1 of DESIGN.md).  One pair at a time, every
 * distance recomputed from the coordinates, no distance vectors kept, no Gram identity: O(L^2) per pair.
 * Inputs are the fp32 arrays the GPU gets, widened to double on load.  L = 1 has no atom pair: returns 0.
 *
 * Pins (tests/test_drmsd_pins.py): identity, rigid copy, MIRROR IMAGE = 0 ("dRMSD ... loses chirality",
 * unlike cRMSD), uniform scaling closed form |1-s| R_g sqrt(2L/(L-1)), two atoms |dA - dB|,
 * scipy pdist route, symmetry and triangle inequality.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (no -ffast-math).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static double dist(const float *x, int i, int j)
{
    double dx = (double)x[3 * i] - (double)x[3 * j];
    double dy = (double)x[3 * i + 1] - (double)x[3 * j + 1];
    double dz = (double)x[3 * i + 2] - (double)x[3 * j + 2];
    return sqrt(dx * dx + dy * dy + dz * dz);
}

/* eq. 5 for one pair; *d2_out (optional) = dRMSD^2 */
double oracle_drmsd_pair(const float *xa, const float *xb, int32_t L, double *d2_out)
{
    double sum = 0.0;
    for (int i = 0; i < L; ++i)
        for (int j = i + 1; j < L; ++j) {
            double diff = dist(xa, i, j) - dist(xb, i, j);
            sum += diff * diff;
        }
    double d2 = L > 1 ? 2.0 * sum / ((double)L * (double)(L - 1)) : 0.0;
    if (d2_out) *d2_out = d2;
    return sqrt(d2);
}

/* Rows [row_begin,row_end) of the packed upper triangle (row-major, j > i), as the cRMSD matrix. */
void oracle_drmsd_rows(const float *coords, int64_t N, int32_t L, int64_t row_begin, int64_t row_end,
                       double *d_out, double *d2_out)
{
    int64_t base = row_begin * (2 * N - row_begin - 1) / 2;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = row_begin; i < row_end; ++i) {
        int64_t off = i * (2 * N - i - 1) / 2 - base;
        for (int64_t j = i + 1; j < N; ++j) {
            double d2;
            d_out[off + (j - i - 1)] = oracle_drmsd_pair(coords + (size_t)i * L * 3, coords + (size_t)j * L * 3, L, &d2);
            if (d2_out) d2_out[off + (j - i - 1)] = d2;
        }
    }
}

/* Listed pairs. */
void oracle_drmsd_pairs(const float *coords, int64_t N, int32_t L, const int64_t *pi, const int64_t *pj,
                        int64_t n_pairs, double *d_out, double *d2_out)
{
    (void)N;
    #pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n_pairs; ++k) {
        double d2;
        d_out[k] = oracle_drmsd_pair(coords + (size_t)pi[k] * L * 3, coords + (size_t)pj[k] * L * 3, L, &d2);
        if (d2_out) d2_out[k] = d2;
    }
}

/* One reference against N models: eq. 5 for (ref, model n). */
void oracle_drmsd_one_vs_all(const float *ref, const float *coords, int64_t N, int32_t L, double *d_out, double *d2_out)
{
    #pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        double d2;
        d_out[n] = oracle_drmsd_pair(ref, coords + (size_t)n * L * 3, L, &d2);
        if (d2_out) d2_out[n] = d2;
    }
}
