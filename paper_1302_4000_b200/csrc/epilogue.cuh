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

    // cofactor rows: C0 = r1 x r2, C1 = r2 x r0, C2 = r0 x r1.  Each entry is a difference of products
    // evaluated with Kahan's FMA scheme (error ~1 ulp of the result): for a rank-deficient M the cofactors
    // are pure cancellation, and det M below inherits their relative accuracy.
    float C[9];
    C[0] = diff_of_products(m[4], m[8], m[5], m[7]);
    C[1] = diff_of_products(m[5], m[6], m[3], m[8]);
    C[2] = diff_of_products(m[3], m[7], m[4], m[6]);
    C[3] = diff_of_products(m[7], m[2], m[8], m[1]);
    C[4] = diff_of_products(m[8], m[0], m[6], m[2]);
    C[5] = diff_of_products(m[6], m[1], m[7], m[0]);
    C[6] = diff_of_products(m[1], m[5], m[2], m[4]);
    C[7] = diff_of_products(m[2], m[3], m[0], m[5]);
    C[8] = diff_of_products(m[0], m[4], m[1], m[3]);
    float c1 = C[0] * C[0];
#pragma unroll
    for (int i = 1; i < 9; ++i) c1 = fmaf(C[i], C[i], c1);
    const float d = fmaf(m[2], C[2], fmaf(m[1], C[1], m[0] * C[0]));     // det M; its sign is S

    EPair r;
    if (!(c2 > 1e-30f)) {                  // M == 0 (L = 1, or every atom on the centroid); NaN passes through
        r.E0 = c2 * 0.0f;                  // 0, or NaN if c2 is NaN
        r.delta = 0.0f;
        return r;
    }

    // largest root of the cubic, Viete:  l1 = q + 2 sqrt(p) cos(acos(rr / p^1.5) / 3)
    const float q = c2 * (1.0f / 3.0f);
    float pp = fmaf(c2, c2, -3.0f * c1) * (1.0f / 9.0f);
    pp = pp > 0.0f ? pp : 0.0f;
    const float d2 = d * d;
    const float rr = fmaf(27.0f, d2, c2 * fmaf(2.0f * c2, c2, -9.0f * c1)) * (1.0f / 54.0f);
    const float sp = sqrtf(pp);
    float ratio = pp > 0.0f ? __fdividef(rr, pp * sp) : 1.0f;
    ratio = fminf(1.0f, fmaxf(-1.0f, ratio));
    const float theta = acosf(ratio) * (1.0f / 3.0f);                   // in [0, pi/3]
    float l1 = fmaf(2.0f * sp, __cosf(theta), q);
    l1 = fmaxf(l1, q);                                                  // l1 >= trace/3 always
    const float s1 = sqrtf(l1);
    const float inv1 = __fdividef(1.0f, l1);
    // deflation: (s2 + S s3)^2 = (c1 - d^2/l1)/l1 + 2 d / s1
    const float w2 = fmaf(2.0f * d, __fdividef(1.0f, s1), (c1 - d2 * inv1) * inv1);
    const float w = sqrtf(w2 > 0.0f ? w2 : 0.0f);
    const float E0 = s1 + w;

    // one Newton step on the quartic; skipped where f' is tiny against E^3 (s2 + S s3 -> 0: the
    // quartic's roots pair up and the deflated value above is the well-conditioned one)
    const float t = fmaf(E0, E0, -c2);
    const float f = fmaf(t, t, fmaf(-8.0f * d, E0, -4.0f * c1));
    const float fp = fmaf(4.0f * E0, t, -8.0f * d);
    r.E0 = E0;
    r.delta = (fp > 1e-3f * E0 * E0 * E0) ? __fdividef(f, fp) : 0.0f;
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

}  // namespace clusco
