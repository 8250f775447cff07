/*
 * gdt_oracle.c -- FP64 CPU oracle for GDT_TS, TM-score and MaxSub of a model against a reference structure.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as crmsd_oracle.c; no code shared with the CUDA path).
 *
 * These three scores are HEURISTICS (the GDT problem is NP-hard), so the oracle follows the paper's
 * algorithm step by step, in the paper's order:
 *
 *   eq. 3   GDT_TS = 1/4 (max C_1A + max C_2A + max C_4A + max C_8A),  C_x = number of atom pairs below x Angstrom,
 *           "Max denotes here the maximal value for a series of superimpositions";
 *   eq. 4   TM-score = max [ 1/N sum_i 1 / (1 + (d_i/d0)^2) ],  d0 = 1.24 cbrt(N - 15) - 1.8;  MaxSub = the same with
 *           d0 = 3.5 A;  "for the calculation of both scores we used the same searching algorithm as for GDT_TS";
 *   search  "1) divide the chain into all possible continuous 4, N/4, N/2, N fragments, and 2) use them as initial
 *           superimposition fragments (i.e. superimpose the whole structure by a rotation matrix computed by
 *           superimposing each fragment), 3) find atom pairs which are closer by cutoff (1, 2, 4, 8 A), 4) select atoms
 *           which are closer than 3.5 A and use them for another superimposition until the number of selected atoms
 *           does not change in four iterations."
 *
 * Readings where the paper is silent: N = number of atoms L; fragment lengths {4, L/4, L/2, L}
 * (integer division, duplicates dropped, lengths below 3 dropped, L < 4 uses {L}); every start 0..L-len; a
 * superposition is the optimal (Kabsch) rigid fit of the model's selected atoms onto the reference's, applied to the
 * whole model; after EVERY superposition (the fragment's and each refinement) all three scores are evaluated and the
 * maxima kept; a refinement needs at least 3 selected atoms; "does not change in four iterations" = the selected
 * count equalled the previous count four times in a row; at most 20 superpositions per fragment; inequalities are
 * strict; GDT_TS is reported as a percentage of L; d0 is clamped at 0.5 A (L <= 21 would make it tiny or negative).
 *
 * The optimal rotation: one-sided Jacobi SVD of the 3x3 covariance matrix of the selected atoms, with the
 * determinant correction for a proper rotation (Kabsch, ref. [1]).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GDT_MAX_ITER 20

/* H = U diag(s) V^T by Hestenes' one-sided Jacobi (columns of W = H V made orthogonal) */
static void svd3(const double H[3][3], double U[3][3], double s[3], double V[3][3])
{
    double W[3][3];
    memcpy(W, H, sizeof W);
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q) V[p][q] = p == q;
    for (int sweep = 0; sweep < 60; ++sweep) {
        int rotated = 0;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                double al = 0, be = 0, ga = 0;
                for (int k = 0; k < 3; ++k) { al += W[k][p] * W[k][p]; be += W[k][q] * W[k][q]; ga += W[k][p] * W[k][q]; }
                if (ga == 0.0 || fabs(ga) <= 1e-15 * sqrt(al * be)) continue;
                rotated = 1;
                double ze = (be - al) / (2.0 * ga);
                double t = (ze >= 0 ? 1.0 : -1.0) / (fabs(ze) + sqrt(1.0 + ze * ze));
                double c = 1.0 / sqrt(1.0 + t * t), sn = c * t;
                for (int k = 0; k < 3; ++k) {
                    double wp = W[k][p], wq = W[k][q], vp = V[k][p], vq = V[k][q];
                    W[k][p] = c * wp - sn * wq; W[k][q] = sn * wp + c * wq;
                    V[k][p] = c * vp - sn * vq; V[k][q] = sn * vp + c * vq;
                }
            }
        if (!rotated) break;
    }
    for (int q = 0; q < 3; ++q) {
        s[q] = sqrt(W[0][q] * W[0][q] + W[1][q] * W[1][q] + W[2][q] * W[2][q]);
        for (int k = 0; k < 3; ++k) U[k][q] = s[q] > 0 ? W[k][q] / s[q] : 0.0;
    }
}

static void cross(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}

/* Optimal proper rotation R and translation t with  a_i ~ R b_i + t  over the atoms with sel[i] != 0. */
static void kabsch(const double *a, const double *b, const unsigned char *sel, int L, double R[3][3], double t[3])
{
    double ca[3] = {0, 0, 0}, cb[3] = {0, 0, 0};
    int n = 0;
    for (int i = 0; i < L; ++i)
        if (sel[i]) { for (int k = 0; k < 3; ++k) { ca[k] += a[3 * i + k]; cb[k] += b[3 * i + k]; } ++n; }
    for (int k = 0; k < 3; ++k) { ca[k] /= n; cb[k] /= n; }
    double H[3][3] = {{0}};                                  /* H = sum (a - ca)(b - cb)^T:  R = U D V^T */
    for (int i = 0; i < L; ++i)
        if (sel[i])
            for (int p = 0; p < 3; ++p)
                for (int q = 0; q < 3; ++q) H[p][q] += (a[3 * i + p] - ca[p]) * (b[3 * i + q] - cb[q]);
    double U[3][3], s[3], V[3][3];
    svd3(H, U, s, V);
    /* take the two leading singular pairs and complete BOTH bases by cross products: both are then right-handed, so
       R = sum u_k v_k^T is a proper rotation -- equal to U diag(1, 1, det(U V^T)) V^T, Kabsch's determinant correction */
    int o[3] = {0, 1, 2};
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2 - i; ++j)
            if (s[o[j]] < s[o[j + 1]]) { int tt = o[j]; o[j] = o[j + 1]; o[j + 1] = tt; }
    double u0[3], u1[3], u2[3], v0[3], v1[3], v2[3];
    for (int k = 0; k < 3; ++k) { u0[k] = U[k][o[0]]; u1[k] = U[k][o[1]]; v0[k] = V[k][o[0]]; v1[k] = V[k][o[1]]; }
    if (u0[0] * u0[0] + u0[1] * u0[1] + u0[2] * u0[2] < 0.5) {   /* H = 0 (all selected atoms coincide): keep the orientation */
        u0[0] = v0[0] = 1.0; u0[1] = u0[2] = v0[1] = v0[2] = 0.0;
        u1[0] = v1[0] = 0.0; u1[1] = v1[1] = 1.0; u1[2] = v1[2] = 0.0;
    }
    /* a rank-1 covariance leaves u1 = 0: complete with any unit vector orthogonal to u0 (the fit is then degenerate) */
    if (u1[0] * u1[0] + u1[1] * u1[1] + u1[2] * u1[2] < 0.5) {
        double e[3] = {0, 0, 0};
        int m = fabs(u0[0]) <= fabs(u0[1]) ? (fabs(u0[0]) <= fabs(u0[2]) ? 0 : 2) : (fabs(u0[1]) <= fabs(u0[2]) ? 1 : 2);
        e[m] = 1.0;
        cross(u0, e, u1);
        double nn = sqrt(u1[0] * u1[0] + u1[1] * u1[1] + u1[2] * u1[2]);
        for (int k = 0; k < 3; ++k) u1[k] /= nn;
    }
    cross(u0, u1, u2);
    cross(v0, v1, v2);                                       /* u2, v2: right-handed completions => det(R) = +1 */
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q) R[p][q] = u0[p] * v0[q] + u1[p] * v1[q] + u2[p] * v2[q];
    for (int p = 0; p < 3; ++p) t[p] = ca[p] - (R[p][0] * cb[0] + R[p][1] * cb[1] + R[p][2] * cb[2]);
}

typedef struct { double c[4]; double tm, maxsub; } gdt_best;

/* evaluate the scores of one superposition (R, t), keep the maxima, and select the atoms closer than 3.5 A */
static int evaluate(const double *a, const double *b, int L, double R[3][3], const double t[3], double d0,
                    gdt_best *best, unsigned char *sel)
{
    static const double cut[4] = {1.0, 2.0, 4.0, 8.0};
    double cnt[4] = {0, 0, 0, 0}, tm = 0.0, ms = 0.0;
    int nsel = 0;
    for (int i = 0; i < L; ++i) {
        double y[3];
        for (int p = 0; p < 3; ++p) y[p] = R[p][0] * b[3 * i] + R[p][1] * b[3 * i + 1] + R[p][2] * b[3 * i + 2] + t[p];
        double dx = a[3 * i] - y[0], dy = a[3 * i + 1] - y[1], dz = a[3 * i + 2] - y[2];
        double d = sqrt(dx * dx + dy * dy + dz * dz);
        for (int c = 0; c < 4; ++c) cnt[c] += d < cut[c];
        tm += 1.0 / (1.0 + (d / d0) * (d / d0));
        ms += 1.0 / (1.0 + (d / 3.5) * (d / 3.5));
        sel[i] = d < 3.5;
        nsel += sel[i];
    }
    for (int c = 0; c < 4; ++c) if (cnt[c] > best->c[c]) best->c[c] = cnt[c];
    if (tm / L > best->tm) best->tm = tm / L;
    if (ms / L > best->maxsub) best->maxsub = ms / L;
    return nsel;
}

/* One model against the reference: out[0] = GDT_TS (percent), out[1] = TM-score, out[2] = MaxSub;
   counts (optional) = max C_1, C_2, C_4, C_8;  trace (optional, diagnostics of the search control only -- no
   arithmetic depends on it): trace[0] = number of seed fragments, trace[1] = superpositions evaluated in total,
   trace[2] = most superpositions spent on one seed. */
void oracle_gdt_pair_trace(const float *ref, const float *model, int32_t L, double *out, double *counts, int64_t *trace)
{
    int64_t n_seeds = 0, n_sup = 0, max_sup = 0;
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)L), *b = (double *)malloc(sizeof(double) * 3 * (size_t)L);
    unsigned char *sel = (unsigned char *)malloc((size_t)L);
    for (int i = 0; i < 3 * L; ++i) { a[i] = ref[i]; b[i] = model[i]; }
    double d0 = 1.24 * cbrt((double)L - 15.0) - 1.8;
    if (!(d0 >= 0.5)) d0 = 0.5;
    gdt_best best = {{0, 0, 0, 0}, 0.0, 0.0};
    int lens[4] = {4, L / 4, L / 2, L}, nl = 0, use[4];
    if (L < 4) { lens[0] = L; use[nl++] = 0; }
    else
        for (int k = 0; k < 4; ++k) {
            int dup = lens[k] < 3;
            for (int m = 0; m < nl; ++m) dup |= lens[use[m]] == lens[k];
            if (!dup) use[nl++] = k;
        }
    for (int m = 0; m < nl; ++m) {
        int len = lens[use[m]];
        for (int start = 0; start + len <= L; ++start) {
            for (int i = 0; i < L; ++i) sel[i] = i >= start && i < start + len;
            int prev = len, same = 0;
            int64_t sup = 0;
            for (int it = 0; it < GDT_MAX_ITER; ++it) {
                double R[3][3], t[3];
                kabsch(a, b, sel, L, R, t);
                int n = evaluate(a, b, L, R, t, d0, &best, sel);
                ++sup;
                if (n == prev) ++same; else same = 0;
                prev = n;
                if (same == 4 || n < 3) break;
            }
            ++n_seeds;
            n_sup += sup;
            if (sup > max_sup) max_sup = sup;
        }
    }
    if (trace) { trace[0] = n_seeds; trace[1] = n_sup; trace[2] = max_sup; }
    out[0] = 100.0 * 0.25 * (best.c[0] + best.c[1] + best.c[2] + best.c[3]) / (double)L;
    out[1] = best.tm;
    out[2] = best.maxsub;
    if (counts) for (int c = 0; c < 4; ++c) counts[c] = best.c[c];
    free(a); free(b); free(sel);
}

void oracle_gdt_pair(const float *ref, const float *model, int32_t L, double *out, double *counts)
{
    oracle_gdt_pair_trace(ref, model, L, out, counts, 0);
}

/* The reference against N models: out[3 n + {0,1,2}]. */
void oracle_gdt_one_vs_all(const float *ref, const float *coords, int64_t N, int32_t L, double *out)
{
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t n = 0; n < N; ++n) oracle_gdt_pair(ref, coords + (size_t)n * L * 3, L, out + 3 * n, 0);
}
