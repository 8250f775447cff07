/*
 * cmo_oracle.c -- FP64 CPU oracle for the Contact Map Overlap (CMO) of protein models.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as crmsd_oracle.c; no code shared with the CUDA path).
 *
 * What it computes: the paper's eq. 6 and eq. 7 written out literally,
 *     C_ij = 1 if |x_i - x_j| < cut-off, 0 otherwise            (eq. 6)
 *     S = 100 * 2 n(A and B) / (n(A) + n(B))                     (eq. 7; n = number of contacts)
 * one pair of models at a time, every contact recomputed from the coordinates: O(L^2) per pair, no stored maps.
 * Readings: contacts are pairs of DISTINCT atoms, counted once (i < j) -- counting both
 * (i,j) and (j,i) gives the same S, counting the diagonal would not; the paper gives no cut-off, so it is an
 * argument; two maps without any contact are identical maps, S = 100 (0/0).
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

static int contact(const float *x, int i, int j, double cutoff)
{
    double dx = (double)x[3 * i] - (double)x[3 * j];
    double dy = (double)x[3 * i + 1] - (double)x[3 * j + 1];
    double dz = (double)x[3 * i + 2] - (double)x[3 * j + 2];
    return sqrt(dx * dx + dy * dy + dz * dz) < cutoff;
}

/* eq. 6-7 for one pair; counts (optional) = {n(A), n(B), n(A and B)} */
double oracle_cmo_pair(const float *xa, const float *xb, int32_t L, double cutoff, int64_t *counts)
{
    int64_t na = 0, nb = 0, nab = 0;
    for (int i = 0; i < L; ++i)
        for (int j = i + 1; j < L; ++j) {
            int ca = contact(xa, i, j, cutoff), cb = contact(xb, i, j, cutoff);
            na += ca;
            nb += cb;
            nab += ca & cb;
        }
    if (counts) { counts[0] = na; counts[1] = nb; counts[2] = nab; }
    if (na + nb == 0) return 100.0;
    return 200.0 * (double)nab / (double)(na + nb);
}

void oracle_cmo_rows(const float *coords, int64_t N, int32_t L, double cutoff, int64_t row_begin, int64_t row_end,
                     double *s_out)
{
    int64_t base = row_begin * (2 * N - row_begin - 1) / 2;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = row_begin; i < row_end; ++i) {
        int64_t off = i * (2 * N - i - 1) / 2 - base;
        for (int64_t j = i + 1; j < N; ++j)
            s_out[off + (j - i - 1)] = oracle_cmo_pair(coords + (size_t)i * L * 3, coords + (size_t)j * L * 3, L, cutoff, 0);
    }
}

void oracle_cmo_pairs(const float *coords, int64_t N, int32_t L, double cutoff, const int64_t *pi, const int64_t *pj,
                      int64_t n_pairs, double *s_out)
{
    (void)N;
    #pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n_pairs; ++k)
        s_out[k] = oracle_cmo_pair(coords + (size_t)pi[k] * L * 3, coords + (size_t)pj[k] * L * 3, L, cutoff, 0);
}

/* One reference against N models: eq. 6-7 for (ref, model n). */
void oracle_cmo_one_vs_all(const float *ref, const float *coords, int64_t N, int32_t L, double cutoff, double *s_out)
{
    #pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) s_out[n] = oracle_cmo_pair(ref, coords + (size_t)n * L * 3, L, cutoff, 0);
}
