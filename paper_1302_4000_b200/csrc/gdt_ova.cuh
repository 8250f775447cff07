// gdt_ova.cuh -- GDT_TS, TM-score and MaxSub of N models against one reference structure (SURVEY.md section 8(f),
// NEXT-4), by the paper's search: every continuous fragment of length 4, L/4, L/2, L seeds a
// superposition; the atoms closer than 3.5 A are re-superposed until their number has not changed in four
// iterations; after every superposition the pair counts below 1, 2, 4, 8 A (eq. 3), the TM-score sum (eq. 4,
// d0 = 1.24 cbrt(L - 15) - 1.8) and the MaxSub sum (d0 = 3.5 A) are evaluated and their maxima kept.
// Readings of the silent points: DESIGN.md section 14 (the same as the oracle's).
//
// The scores are heuristic maxima over a data-dependent series of superpositions, so everything is FP64: a distance
// on the wrong side of a cut-off would change the series.  One warp per model, lane = atoms lane, lane + 32, ...;
// selections are per-lane bit masks.  Per superposition: 16 warp-reduced sums (count, two centroids, the 3x3
// cross-covariance of the selected atoms) -> every lane computes the optimal proper rotation redundantly by HORN'S
// QUATERNION route -- the largest eigenvalue of the 4x4 key matrix is the largest root of the quartic
// (E^2 - c2)^2 - 8 d E - 4 c1 = 0 (c2 = |H|_F^2, c1 = |cof H|_F^2, d = det H), found by Newton's iteration from the
// upper bound sqrt(3 c2); its eigenvector is the best-conditioned column of adj(N - E I) -- no SVD, no Jacobi sweeps
// (the oracle uses a Jacobi SVD: the two routes share nothing).
#pragma once
#include "common.cuh"
#include "prep.cuh"

namespace clusco {

constexpr int GDT_WARPS = 4;
constexpr int GDT_MAX_L = 1024;                // 32 mask bits per lane
constexpr int GDT_MAX_ITER = 20;

__device__ __forceinline__ double gdt_det3(double a, double b, double c, double d, double e, double f, double g, double h,
                                           double i)
{
    return a * (e * i - f * h) - b * (d * i - f * g) + c * (d * h - e * g);
}

// Proper rotation R (row-major) with  target ~ R model  from S[p][q] = sum model_p target_q (centred on the selection).
__device__ __forceinline__ void gdt_rotation(const double S[9], double R[9])
{
    const double Sxx = S[0], Sxy = S[1], Sxz = S[2], Syx = S[3], Syy = S[4], Syz = S[5], Szx = S[6], Szy = S[7], Szz = S[8];
    // invariants of the quartic
    double c2 = 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) c2 += S[k] * S[k];
    const double C00 = Syy * Szz - Syz * Szy, C01 = Syz * Szx - Syx * Szz, C02 = Syx * Szy - Syy * Szx;
    const double C10 = Sxz * Szy - Sxy * Szz, C11 = Sxx * Szz - Sxz * Szx, C12 = Sxy * Szx - Sxx * Szy;
    const double C20 = Sxy * Syz - Sxz * Syy, C21 = Sxz * Syx - Sxx * Syz, C22 = Sxx * Syy - Sxy * Syx;
    const double c1 = C00 * C00 + C01 * C01 + C02 * C02 + C10 * C10 + C11 * C11 + C12 * C12 + C20 * C20 + C21 * C21 + C22 * C22;
    const double d = Sxx * C00 + Sxy * C01 + Sxz * C02;
    R[0] = R[4] = R[8] = 1.0;
    R[1] = R[2] = R[3] = R[5] = R[6] = R[7] = 0.0;
    if (!(c2 > 0.0)) return;                                     // no spread at all: keep the orientation
    // largest root by Newton from above (f is increasing and convex to the right of its largest root)
    double E = sqrt(3.0 * c2);
    for (int it = 0; it < 100; ++it) {
        const double t = E * E - c2;
        const double f = t * t - 8.0 * d * E - 4.0 * c1;
        const double fp = 4.0 * E * t - 8.0 * d;
        if (!(fp > 0.0)) break;
        const double step = f / fp;
        E -= step;
        if (fabs(step) <= 1e-15 * E) break;
    }
    // key matrix N - E I (symmetric); its adjugate is (a multiple of) q q^T, q the top eigenvector
    double M[4][4];
    M[0][0] = Sxx + Syy + Szz - E; M[0][1] = Syz - Szy; M[0][2] = Szx - Sxz; M[0][3] = Sxy - Syx;
    M[1][1] = Sxx - Syy - Szz - E; M[1][2] = Sxy + Syx; M[1][3] = Szx + Sxz;
    M[2][2] = -Sxx + Syy - Szz - E; M[2][3] = Syz + Szy;
    M[3][3] = -Sxx - Syy + Szz - E;
#pragma unroll
    for (int r = 1; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < r; ++c) M[r][c] = M[c][r];
    double adj[4][4];                                            // all 16 cofactors (compile-time indices: registers only)
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = r; c < 4; ++c) {
            const int r0 = r == 0 ? 1 : 0, r1 = r <= 1 ? 2 : 1, r2 = r <= 2 ? 3 : 2;
            const int k0 = c == 0 ? 1 : 0, k1 = c <= 1 ? 2 : 1, k2 = c <= 2 ? 3 : 2;
            const double m = gdt_det3(M[r0][k0], M[r0][k1], M[r0][k2], M[r1][k0], M[r1][k1], M[r1][k2], M[r2][k0], M[r2][k1],
                                      M[r2][k2]);
            adj[r][c] = adj[c][r] = ((r + c) & 1) ? -m : m;
        }
    // the best-conditioned column: the one with the largest diagonal entry (= c q_k^2)
    int j = 0;
    double best = fabs(adj[0][0]);
#pragma unroll
    for (int k = 1; k < 4; ++k)
        if (fabs(adj[k][k]) > best) { best = fabs(adj[k][k]); j = k; }
    double q0 = adj[0][0], q1 = adj[1][0], q2 = adj[2][0], q3 = adj[3][0];
#pragma unroll
    for (int k = 1; k < 4; ++k)
        if (j == k) { q0 = adj[0][k]; q1 = adj[1][k]; q2 = adj[2][k]; q3 = adj[3][k]; }
    const double nn = q0 * q0 + q1 * q1 + q2 * q2 + q3 * q3;
    if (!(nn > 0.0)) return;                                     // degenerate (double top eigenvalue): keep the orientation
    const double inv = 1.0 / sqrt(nn);
    q0 *= inv; q1 *= inv; q2 *= inv; q3 *= inv;
    R[0] = q0 * q0 + q1 * q1 - q2 * q2 - q3 * q3; R[1] = 2.0 * (q1 * q2 - q0 * q3); R[2] = 2.0 * (q1 * q3 + q0 * q2);
    R[3] = 2.0 * (q1 * q2 + q0 * q3); R[4] = q0 * q0 - q1 * q1 + q2 * q2 - q3 * q3; R[5] = 2.0 * (q2 * q3 - q0 * q1);
    R[6] = 2.0 * (q1 * q3 - q0 * q2); R[7] = 2.0 * (q2 * q3 + q0 * q1); R[8] = q0 * q0 - q1 * q1 - q2 * q2 + q3 * q3;
}

// 1 / x for x >= 1: fp32 reciprocal seed + two FP64 Newton steps (relative error ~1e-15; an IEEE division is ~4x the work)
__device__ __forceinline__ double gdt_rcp(double x)
{
    double y = (double)__frcp_rn((float)x);
    y = y * (2.0 - x * y);
    y = y * (2.0 - x * y);
    return y;
}

__device__ __forceinline__ double gdt_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sums of 16 values over the warp, every lane receiving all 16: a transposed butterfly -- at offset 16 a lane keeps one
// half of the values and hands the other half to its partner, at offset 8 a quarter, ... -- so that 16 exchanges (plus 16
// broadcasts) replace the 80 of sixteen separate butterflies.  Value e ends up on lanes 2 e and 2 e + 1.
__device__ __forceinline__ void gdt_warp_sum16(double (&v)[16], int lane)
{
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4, b1 = lane & 2;
    double w8[8], w4[4], w2[2];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        const double keep = b4 ? v[e + 8] : v[e], send = b4 ? v[e] : v[e + 8];
        w8[e] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const double keep = b3 ? w8[e + 4] : w8[e], send = b3 ? w8[e] : w8[e + 4];
        w4[e] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const double keep = b2 ? w4[e + 2] : w4[e], send = b2 ? w4[e] : w4[e + 2];
        w2[e] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    double w1 = (b1 ? w2[1] : w2[0]) + __shfl_xor_sync(0xffffffffu, b1 ? w2[0] : w2[1], 2);
    w1 += __shfl_xor_sync(0xffffffffu, w1, 1);
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = __shfl_sync(0xffffffffu, w1, 2 * e);
}

// centre a model (FP64) into shared memory, one warp; returns whether all its coordinates are finite
__device__ __forceinline__ bool gdt_load_centred(double* __restrict__ dst, const float* __restrict__ x, int L, int lane)
{
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    bool fin = true;
    for (int i = lane; i < L; i += 32) {
        const float v0 = x[3 * i], v1 = x[3 * i + 1], v2 = x[3 * i + 2];
        fin = fin && fabsf(v0) <= 3.0e38f && fabsf(v1) <= 3.0e38f && fabsf(v2) <= 3.0e38f;
        s0 += (double)v0; s1 += (double)v1; s2 += (double)v2;
    }
    s0 = gdt_warp_sum(s0) / (double)L; s1 = gdt_warp_sum(s1) / (double)L; s2 = gdt_warp_sum(s2) / (double)L;
    fin = __all_sync(0xffffffffu, fin);
    __syncwarp();
    for (int i = lane; i < L; i += 32) {
        dst[3 * i] = (double)x[3 * i] - s0; dst[3 * i + 1] = (double)x[3 * i + 1] - s1; dst[3 * i + 2] = (double)x[3 * i + 2] - s2;
    }
    __syncwarp();
    return fin;
}

// out[3 n + {0, 1, 2}] = GDT_TS (percent), TM-score, MaxSub of model n against the reference.
// Dynamic shared memory: (1 + GDT_WARPS) * 3 L doubles -- the reference and one model per warp, each centred on its own
// centroid (rigid motions do not change the scores; centring keeps the covariance sums free of cancellation).
// ALLPAIRS: unit = pair (i < j) of the packed upper triangle, reference = model i (the search is symmetric in the two
// structures: selections depend on distances only), out[3 idx + ...] with idx the packed index; both models per warp.
template <bool ALLPAIRS>
__global__ void __launch_bounds__(GDT_WARPS * 32) gdt_kernel(const float* __restrict__ ref, const float* __restrict__ coords,
                                                             int64_t N, int32_t L, float* __restrict__ out)
{
    extern __shared__ __align__(16) double gdt_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* A = ALLPAIRS ? gdt_smem + (size_t)(2 * warp) * 3 * L : gdt_smem;                       // reference, 3 L
    double* B = ALLPAIRS ? gdt_smem + (size_t)(2 * warp + 1) * 3 * L : gdt_smem + (size_t)(1 + warp) * 3 * L;
    // one-vs-all: every CTA centres the reference itself (FP64)
    if (!ALLPAIRS) {
        __shared__ double red[3][GDT_WARPS];
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
        for (int i = threadIdx.x; i < L; i += blockDim.x) { s0 += (double)ref[3 * i]; s1 += (double)ref[3 * i + 1]; s2 += (double)ref[3 * i + 2]; }
        s0 = gdt_warp_sum(s0); s1 = gdt_warp_sum(s1); s2 = gdt_warp_sum(s2);
        if (lane == 0) { red[0][warp] = s0; red[1][warp] = s1; red[2][warp] = s2; }
        __syncthreads();
        double m[3] = {0.0, 0.0, 0.0};
        for (int w = 0; w < GDT_WARPS; ++w) { m[0] += red[0][w]; m[1] += red[1][w]; m[2] += red[2][w]; }
        for (int e = threadIdx.x; e < 3 * L; e += blockDim.x) A[e] = (double)ref[e] - m[e % 3] / (double)L;
        __syncthreads();
    }
    double d0 = 1.24 * cbrt((double)L - 15.0) - 1.8;
    if (!(d0 >= 0.5)) d0 = 0.5;
    const double inv_d0sq = 1.0 / (d0 * d0), inv_35sq = 1.0 / (3.5 * 3.5);
    const int nk = (L + 31) >> 5;                                // atoms per lane (mask bits)
    int lens[4] = {4, L / 4, L / 2, L};
    if (L < 4) lens[0] = lens[1] = lens[2] = L;

    const int64_t total = ALLPAIRS ? N * (N - 1) / 2 : N;
    for (int64_t n = (int64_t)blockIdx.x * GDT_WARPS + warp; n < total; n += (int64_t)gridDim.x * GDT_WARPS) {
        bool finite = true;
        int64_t jm = n;                                          // the model superposed onto the reference
        if (ALLPAIRS) {
            // packed index n -> (i, j): row i starts at i (2N - i - 1) / 2
            const double Nd = (double)N;
            int64_t i = (int64_t)floor(((2.0 * Nd - 1.0) - sqrt((2.0 * Nd - 1.0) * (2.0 * Nd - 1.0) - 8.0 * (double)n)) * 0.5);
            if (i < 0) i = 0;
            while (i > 0 && i * (2 * N - i - 1) / 2 > n) --i;
            while ((i + 1) * (2 * N - i - 2) / 2 <= n) ++i;
            jm = i + 1 + (n - i * (2 * N - i - 1) / 2);
            finite = gdt_load_centred(A, coords + i * (int64_t)L * 3, L, lane);
        }
        finite = gdt_load_centred(B, coords + jm * (int64_t)L * 3, L, lane) && finite;
        int bestc0 = 0, bestc1 = 0, bestc2 = 0, bestc3 = 0;
        double best_tm = 0.0, best_ms = 0.0;
        for (int f = 0; f < 4; ++f) {
            const int len = lens[f];
            bool dup = len < 3 && !(L < 4 && f == 0);
            for (int g = 0; g < f; ++g) dup = dup || lens[g] == len;
            if (dup) continue;                                   // warp-uniform
            for (int start = 0; start + len <= L; ++start) {
                uint32_t mask = 0u;                              // bit k: atom lane + 32 k selected
                for (int k = 0; k < nk; ++k) {
                    const int i = lane + 32 * k;
                    if (i >= start && i < start + len) mask |= 1u << k;
                }
                int prev = len, same = 0;
                for (int it = 0; it < GDT_MAX_ITER; ++it) {
                    // sums over the selected atoms
                    double cnt = 0.0, ca0 = 0.0, ca1 = 0.0, ca2 = 0.0, cb0 = 0.0, cb1 = 0.0, cb2 = 0.0;
                    double S[9] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
                    for (int k = 0; k < nk; ++k)
                        if (mask >> k & 1u) {
                            const int i = lane + 32 * k;
                            const double a0 = A[3 * i], a1 = A[3 * i + 1], a2 = A[3 * i + 2];
                            const double b0 = B[3 * i], b1 = B[3 * i + 1], b2 = B[3 * i + 2];
                            cnt += 1.0;
                            ca0 += a0; ca1 += a1; ca2 += a2; cb0 += b0; cb1 += b1; cb2 += b2;
                            S[0] += b0 * a0; S[1] += b0 * a1; S[2] += b0 * a2;
                            S[3] += b1 * a0; S[4] += b1 * a1; S[5] += b1 * a2;
                            S[6] += b2 * a0; S[7] += b2 * a1; S[8] += b2 * a2;
                        }
                    {
                        double v[16] = {cnt, ca0, ca1, ca2, cb0, cb1, cb2, S[0], S[1], S[2], S[3], S[4], S[5], S[6], S[7], S[8]};
                        gdt_warp_sum16(v, lane);
                        cnt = v[0];
                        ca0 = v[1] / cnt; ca1 = v[2] / cnt; ca2 = v[3] / cnt;
                        cb0 = v[4] / cnt; cb1 = v[5] / cnt; cb2 = v[6] / cnt;
#pragma unroll
                        for (int e = 0; e < 9; ++e) S[e] = v[7 + e];
                    }
                    // centre the cross-covariance on the selection: S - n cb ca^T
                    S[0] -= cnt * cb0 * ca0; S[1] -= cnt * cb0 * ca1; S[2] -= cnt * cb0 * ca2;
                    S[3] -= cnt * cb1 * ca0; S[4] -= cnt * cb1 * ca1; S[5] -= cnt * cb1 * ca2;
                    S[6] -= cnt * cb2 * ca0; S[7] -= cnt * cb2 * ca1; S[8] -= cnt * cb2 * ca2;
                    double R[9];
                    gdt_rotation(S, R);
                    const double t0 = ca0 - (R[0] * cb0 + R[1] * cb1 + R[2] * cb2);
                    const double t1 = ca1 - (R[3] * cb0 + R[4] * cb1 + R[5] * cb2);
                    const double t2 = ca2 - (R[6] * cb0 + R[7] * cb1 + R[8] * cb2);
                    // evaluate this superposition on all atoms
                    int c0 = 0, c1 = 0, c2 = 0, c3 = 0, nsel = 0;
                    double tm = 0.0, ms = 0.0;
                    mask = 0u;
                    for (int k = 0; k < nk; ++k) {
                        const int i = lane + 32 * k;
                        if (i < L) {
                            const double b0 = B[3 * i], b1 = B[3 * i + 1], b2 = B[3 * i + 2];
                            const double dx = A[3 * i] - (R[0] * b0 + R[1] * b1 + R[2] * b2 + t0);
                            const double dy = A[3 * i + 1] - (R[3] * b0 + R[4] * b1 + R[5] * b2 + t1);
                            const double dz = A[3 * i + 2] - (R[6] * b0 + R[7] * b1 + R[8] * b2 + t2);
                            const double dd = dx * dx + dy * dy + dz * dz;
                            // d < x decided as d^2 < x^2 (x^2 exact in FP64; differs from comparing the rounded square root
                            // only for d^2 within one ulp of x^2), no square root per atom
                            c0 += dd < 1.0; c1 += dd < 4.0; c2 += dd < 16.0; c3 += dd < 64.0;
                            tm += gdt_rcp(1.0 + dd * inv_d0sq);
                            ms += gdt_rcp(1.0 + dd * inv_35sq);
                            if (dd < 12.25) { mask |= 1u << k; ++nsel; }
                        }
                    }
                    c0 = __reduce_add_sync(0xffffffffu, c0); c1 = __reduce_add_sync(0xffffffffu, c1);
                    c2 = __reduce_add_sync(0xffffffffu, c2); c3 = __reduce_add_sync(0xffffffffu, c3);
                    nsel = __reduce_add_sync(0xffffffffu, nsel);
                    tm = gdt_warp_sum(tm) / (double)L;
                    ms = gdt_warp_sum(ms) / (double)L;
                    bestc0 = max(bestc0, c0); bestc1 = max(bestc1, c1); bestc2 = max(bestc2, c2); bestc3 = max(bestc3, c3);
                    best_tm = fmax(best_tm, tm);
                    best_ms = fmax(best_ms, ms);
                    if (nsel == prev) ++same; else same = 0;
                    prev = nsel;
                    if (same == 4 || nsel < 3) break;
                }
            }
        }
        if (lane == 0) {
            const float nanv = __int_as_float(0x7fc00000);
            out[3 * n] = finite ? (float)(100.0 * 0.25 * (double)(bestc0 + bestc1 + bestc2 + bestc3) / (double)L) : nanv;
            out[3 * n + 1] = finite ? (float)best_tm : nanv;
            out[3 * n + 2] = finite ? (float)best_ms : nanv;
        }
        __syncwarp();
    }
}

}  // namespace clusco
