// epilogue.cuh -- per-pair closed form of the paper's eq. 2, shared by every kernel.
//
// Input: the nine entries of a pair's 3x3 covariance matrix M (any common scale; the callers pass the
// unnormalised Gram sums of power-of-two-scaled centred coordinates).  Output: E = s1 + s2 + S*s3, the
// quantity eq. 2 writes as sqrt(l1)+sqrt(l2)+S*sqrt(l3) with l_k the descending eigenvalues of M^T M
// ("the square of the covariance matrix") and S = sign det M -- found from the CUBIC characteristic
// polynomial of M^T M, with no SVD and no rotation matrix.
//
// How:  the cubic  l^3 - c2 l^2 + c1 l - d^2 = 0  has coefficients
//     c2 = |M|_F^2,  c1 = |cof M|_F^2,  d = det M
// taken from M itself (never from an explicitly squared matrix, which would square the condition
// number).  Only the LARGEST root l1 is taken from Viete's trigonometric formula; the two small ones are
// deflated out:   l2 + l3 = (c1 - d^2/l1)/l1,   sqrt(l2 l3) = |d|/s1,   so
//     (s2 + S s3)^2 = l2 + l3 + 2 d / s1          -- S enters through the sign of d, exactly as eq. 2 says.
// That value E0 is then polished by one Newton step on the quartic E satisfies,
//     f(E) = (E^2 - c2)^2 - 8 d E - 4 c1 = 0,     f'(E) = 4 E (E^2 - c2) - 8 d,
// and returned as the unevaluated pair (E0, delta), E = E0 - delta, so that the caller's final
// R_A^2 + R_B^2 - 2E cancels without rounding E first.
#pragma once
#include "common.cuh"

namespace clusco {

struct EPair { float E0; float delta; };

// ---- fast single-instruction approximations (MUFU), relative error ~2^-22; every use below is either polished
// by the Newton step that follows or far inside the output tolerance ---------------------------------------
__device__ __forceinline__ float rcp_fast(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_fast(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_fast(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float cos_fast(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// acos on [-1, 1]: sqrt(1 - |x|) * P7(|x|)  (Abramowitz & Stegun 4.4.46, |error| <= 2e-8), reflected for x < 0
__device__ __forceinline__ float acos_fast(float x)
{
    const float ax = fabsf(x);
    float p = -0.0012624911f;
    p = fmaf(p, ax, 0.0066700901f);
    p = fmaf(p, ax, -0.0170881256f);
    p = fmaf(p, ax, 0.0308918810f);
    p = fmaf(p, ax, -0.0501743046f);
    p = fmaf(p, ax, 0.0889789874f);
    p = fmaf(p, ax, -0.2145988016f);
    p = fmaf(p, ax, 1.5707963050f);
    const float r = sqrt_fast(1.0f - ax) * p;
    return x < 0.0f ? 3.14159265358979f - r : r;
}

// a*b - c*d with one rounding error of the result (Kahan): w = c*d rounded, e = exact error of w
__device__ __forceinline__ float diff_of_products(float a, float b, float c, float d)
{
    const float w = c * d;
    const float e = fmaf(-c, d, w);
    const float f = fmaf(a, b, -w);
    return f + e;
}

__device__ __forceinline__ EPair eq2_energy(const float m[9])
{
    // c2 = |M|_F^2
    float c2 = m[0] * m[0];
#pragma unroll
    for (int i = 1; i < 9; ++i) c2 = fmaf(m[i], m[i], c2);

    // cofactor rows: C0 = r1 x r2, C1 = r2 x r0, C2 = r0 x r1.  The first row, which det M is expanded along,
    // uses Kahan's FMA difference of products (error ~1 ulp of the result): for a rank-deficient M the
    // cofactors are pure cancellation and det M must inherit their RELATIVE accuracy, because it enters E
    // under a square root (2 d / s1 below).  The other six only enter through c1 = sum C^2, where an
    // absolute error of eps |M|^2 is harmless.
    float C[9];
    C[0] = diff_of_products(m[4], m[8], m[5], m[7]);
    C[1] = diff_of_products(m[5], m[6], m[3], m[8]);
    C[2] = diff_of_products(m[3], m[7], m[4], m[6]);
    C[3] = fmaf(m[7], m[2], -(m[8] * m[1]));
    C[4] = fmaf(m[8], m[0], -(m[6] * m[2]));
    C[5] = fmaf(m[6], m[1], -(m[7] * m[0]));
    C[6] = fmaf(m[1], m[5], -(m[2] * m[4]));
    C[7] = fmaf(m[2], m[3], -(m[0] * m[5]));
    C[8] = fmaf(m[0], m[4], -(m[1] * m[3]));
    float c1 = C[0] * C[0];
#pragma unroll
    for (int i = 1; i < 9; ++i) c1 = fmaf(C[i], C[i], c1);
    const float d = fmaf(m[2], C[2], fmaf(m[1], C[1], m[0] * C[0]));     // det M; its sign is S

    EPair r;

    // largest root of the cubic, Viete:  l1 = q + 2 sqrt(p) cos(acos(rr / p^1.5) / 3)
    const float q = c2 * (1.0f / 3.0f);
    float pp = fmaf(c2, c2, -3.0f * c1) * (1.0f / 9.0f);
    pp = pp > 0.0f ? pp : 0.0f;
    const float d2 = d * d;
    const float rr = fmaf(27.0f, d2, c2 * fmaf(2.0f * c2, c2, -9.0f * c1)) * (1.0f / 54.0f);
    const float sp = sqrt_fast(pp);
    float ratio = pp > 0.0f ? rr * rcp_fast(pp * sp) : 1.0f;
    ratio = fminf(1.0f, fmaxf(-1.0f, ratio));
    const float theta = acos_fast(ratio) * (1.0f / 3.0f);              // in [0, pi/3]
    float l1 = fmaf(2.0f * sp, cos_fast(theta), q);
    l1 = fmaxf(l1, q);                                                  // l1 >= trace/3 always
    const float is1 = rsqrt_fast(l1);
    const float s1 = l1 * is1;
    const float inv1 = is1 * is1;
    // deflation: (s2 + S s3)^2 = (c1 - d^2/l1)/l1 + 2 d / s1
    const float w2 = fmaf(2.0f * d, is1, (c1 - d2 * inv1) * inv1);
    const float w = sqrt_fast(w2 > 0.0f ? w2 : 0.0f);
    const float E0 = s1 + w;

    // one Newton step on the quartic; skipped where f' is tiny against E^3 (s2 + S s3 -> 0: the
    // quartic's roots pair up and the deflated value above is the well-conditioned one)
    const float t = fmaf(E0, E0, -c2);
    const float f = fmaf(t, t, fmaf(-8.0f * d, E0, -4.0f * c1));
    const float fp = fmaf(4.0f * E0, t, -8.0f * d);
    // M == 0 (L = 1, or every atom on the centroid): E = 0 (the lines above then hold 0 * inf, selected away
    // here, so the function stays branch-free); a NaN in M gives c2 = NaN and passes through as NaN
    const bool nonzero = c2 > 1e-30f;
    r.E0 = nonzero ? E0 : c2 * 0.0f;
    r.delta = (nonzero && fp > 1e-3f * E0 * E0 * E0) ? f * rcp_fast(fp) : 0.0f;
    return r;
}

// The last line of eq. 2 for a pair (i, j) whose models carry power-of-two scales 2^ei, 2^ej:
//   m[] holds the Gram sums of the SCALED coordinates, (Shi,Slo) the two-float sums of squares of the
//   scaled coordinates, so   L c^2 2^-(ei+ej) = S_i 2^(ei-ej) + S_j 2^(ej-ei) - 2 E   with every scaling exact.
__device__ __forceinline__ float eq2_crmsd(const float m[9], float Shi_i, float Slo_i, int ei,
                                           float Shi_j, float Slo_j, int ej, float invL)
{
    const EPair e = eq2_energy(m);
    const int de = max(-60, min(60, ei - ej));
    const float pu = pow2i(de), pv = pow2i(-de);
    // (u - E0) + (v - E0) is exact (Sterbenz) whenever the two models are similar -- exactly when it matters
    float res = (fmaf(Shi_i, pu, -e.E0) + fmaf(Shi_j, pv, -e.E0))
              + fmaf(2.0f, e.delta, fmaf(Slo_i, pu, Slo_j * pv));
    res = res < 0.0f ? 0.0f : res;                                      // clamp (NaN stays NaN)
    const int es = max(-120, min(120, ei + ej));
    return sqrtf(res * invL * pow2i(es - es / 2) * pow2i(es / 2));
}

// The same last line when each model carries T = sum |a|^2 in its TRUE scale as two floats (Thi, Tlo) and
// pw = 2^e (|e| <= 30, so every product below stays far inside the fp32 range):  with pp = pw_i pw_j,
//   L c^2 = (T_i - E pp) + (T_j - E pp);   E0 pp is exact, and each difference is exact by Sterbenz when the
// models are similar.  c = sqrt(max(0, .) / L) by the MUFU square root (relative error 2^-22 << 1e-3 A).
__device__ __forceinline__ float eq2_finish(const EPair e, float Thi_i, float Tlo_i, float pw_i, float Thi_j,
                                            float Tlo_j, float pw_j, float invL)
{
    const float pp = pw_i * pw_j;
    const float E0p = e.E0 * pp;
    float res = ((Thi_i - E0p) + (Thi_j - E0p)) + fmaf(2.0f * e.delta, pp, Tlo_i + Tlo_j);
    res = res < 0.0f ? 0.0f : res;                                      // clamp (NaN stays NaN)
    return sqrt_fast(res * invL);
}

}  // namespace clusco
