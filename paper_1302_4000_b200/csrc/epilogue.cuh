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

// ---- fast single-instruction approximations (MUFU), relative error ~2^-22; every use below is either polished
// by the Newton step that follows or far inside the output tolerance ---------------------------------------
__device__ __forceinline__ float rcp_fast(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_fast(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_fast(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// ---- the arithmetic of the closed form, written once for V = float (one pair per thread) and V = float2 (two
// pairs per thread, evaluated together on the packed FFMA2 / FMUL2 / FADD2 instructions of sm_100; operand
// negation and scalar broadcast fold into those instructions).  Comparisons, selects and MUFU stay per lane. ---
namespace lp {
template <class V> __device__ __forceinline__ V splat(float s);
template <> __device__ __forceinline__ float splat<float>(float s) { return s; }
template <> __device__ __forceinline__ float2 splat<float2>(float s) { return make_float2(s, s); }

__device__ __forceinline__ float fma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float2 fma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float mul(float a, float b) { return a * b; }
__device__ __forceinline__ float2 mul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float add(float a, float b) { return a + b; }
__device__ __forceinline__ float2 add(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float neg(float a) { return -a; }
__device__ __forceinline__ float2 neg(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float sub(float a, float b) { return a - b; }
__device__ __forceinline__ float2 sub(float2 a, float2 b) { return __fadd2_rn(a, neg(b)); }
// per-lane map / zip for the operations that have no packed form
template <class F> __device__ __forceinline__ float map(float a, F f) { return f(a); }
template <class F> __device__ __forceinline__ float2 map(float2 a, F f) { return make_float2(f(a.x), f(a.y)); }
template <class F> __device__ __forceinline__ float zip(float a, float b, F f) { return f(a, b); }
template <class F> __device__ __forceinline__ float2 zip(float2 a, float2 b, F f) { return make_float2(f(a.x, b.x), f(a.y, b.y)); }
template <class F> __device__ __forceinline__ float zip3(float a, float b, float c, F f) { return f(a, b, c); }
template <class F> __device__ __forceinline__ float2 zip3(float2 a, float2 b, float2 c, F f)
{
    return make_float2(f(a.x, b.x, c.x), f(a.y, b.y, c.y));
}
}  // namespace lp

template <class V> struct EPairT { V E0; V delta; };
typedef EPairT<float> EPair;

// cos(acos(x) / 3) on [-1, 1] (Viete's angle trisection) without the angle: with s = sqrt((1 + x) / 2) the
// function is analytic on the whole of [0, 1] (the square-root branch point at x = -1 is absorbed by s, and at
// x = +1 it is even in the angle), so one MUFU square root and a degree-7 minimax polynomial in s give it to
// 1.3e-7 in fp32 Horner arithmetic (fitted on Chebyshev nodes against the FP64 definition).  x outside [-1, 1]
// (rounding) is clamped by the saturating FMA.
template <class V>
__device__ __forceinline__ V cos_third_acos(V x)
{
    using namespace lp;
    const V sv = map(x, [](float t) { return sqrt_fast(__saturatef(fmaf(t, 0.5f, 0.5f))); });
    V p = splat<V>(1.1504285912e-03f);
    p = fma(p, sv, splat<V>(-6.1699481236e-03f));
    p = fma(p, sv, splat<V>(1.6159486845e-02f));
    p = fma(p, sv, splat<V>(-3.0313061318e-02f));
    p = fma(p, sv, splat<V>(5.2869105217e-02f));
    p = fma(p, sv, splat<V>(-1.1104323939e-01f));
    p = fma(p, sv, splat<V>(5.7734722249e-01f));
    p = fma(p, sv, splat<V>(5.0000002277e-01f));
    return p;
}

// a*b - c*d with one rounding error of the result (Kahan): w = c*d rounded, e = exact error of w
template <class V>
__device__ __forceinline__ V diff_of_products(V a, V b, V c, V d)
{
    using namespace lp;
    const V w = mul(c, d);
    const V e = fma(neg(c), d, w);
    const V f = fma(a, b, neg(w));
    return add(f, e);
}

// The three invariants of M the cubic and the quartic are built from: c2 = |M|_F^2, c1 = |cof M|_F^2, d = det M.
template <class V> struct EqInvariants { V c2, c1, d; };

template <class V>
__device__ __forceinline__ EqInvariants<V> eq2_invariants(const V m[9])
{
    using namespace lp;
    // c2 = |M|_F^2
    V c2 = mul(m[0], m[0]);
#pragma unroll
    for (int i = 1; i < 9; ++i) c2 = fma(m[i], m[i], c2);

    // cofactor rows: C0 = r1 x r2, C1 = r2 x r0, C2 = r0 x r1.  The first row, which det M is expanded along,
    // uses Kahan's FMA difference of products (error ~1 ulp of the result): for a rank-deficient M the
    // cofactors are pure cancellation and det M must inherit their RELATIVE accuracy, because it enters E
    // under a square root (2 d / s1 below).  The other six only enter through c1 = sum C^2, where an
    // absolute error of eps |M|^2 is harmless.
    V C[9];
    C[0] = diff_of_products(m[4], m[8], m[5], m[7]);
    C[1] = diff_of_products(m[5], m[6], m[3], m[8]);
    C[2] = diff_of_products(m[3], m[7], m[4], m[6]);
    C[3] = fma(m[7], m[2], neg(mul(m[8], m[1])));
    C[4] = fma(m[8], m[0], neg(mul(m[6], m[2])));
    C[5] = fma(m[6], m[1], neg(mul(m[7], m[0])));
    C[6] = fma(m[1], m[5], neg(mul(m[2], m[4])));
    C[7] = fma(m[2], m[3], neg(mul(m[0], m[5])));
    C[8] = fma(m[0], m[4], neg(mul(m[1], m[3])));
    V c1 = mul(C[0], C[0]);
#pragma unroll
    for (int i = 1; i < 9; ++i) c1 = fma(C[i], C[i], c1);
    EqInvariants<V> r;
    r.c2 = c2;
    r.c1 = c1;
    r.d = fma(m[2], C[2], fma(m[1], C[1], mul(m[0], C[0])));           // det M; its sign is S
    return r;
}

// E from the invariants (the serial, latency-bound half of the closed form; the tensor-core engine overlaps it
// with the next tile's accumulator loads)
template <class V>
__device__ __forceinline__ EPairT<V> eq2_energy(const EqInvariants<V> inv)
{
    using namespace lp;
    const V c2 = inv.c2, c1 = inv.c1, d = inv.d;
    // largest root of the cubic, Viete:  l1 = q + 2 sqrt(p) cos(acos(rr / p^1.5) / 3)
    // with q = c2 / 3:  p = (c2^2 - 3 c1) / 9 = q^2 - c1 / 3,   r = (27 d^2 + c2 (2 c2^2 - 9 c1)) / 54 = d^2 / 2 + q (q^2 - c1 / 2)
    // p is kept away from zero (three equal roots, or M == 0) by a floor far below anything that matters; 1 / sqrt(p)
    // then serves both sqrt(p) and p^-1.5.  Where p sits on the floor the ratio may overflow or be 0 * inf: the saturating
    // FMA inside cos_third_acos maps +-inf to 0 / 1 and NaN to 0, and the factor sqrt(p) ~ 1e-15 makes the term vanish.
    const V q = mul(c2, splat<V>(1.0f / 3.0f));
    const V qq = mul(q, q);
    const V pp = map(fma(c1, splat<V>(-1.0f / 3.0f), qq), [](float t) { return fmaxf(t, 1e-30f); });
    const V isp = map(pp, [](float t) { return rsqrt_fast(t); });
    const V sp = mul(pp, isp);
    const V d2 = mul(d, d);
    const V rr = fma(q, fma(c1, splat<V>(-0.5f), qq), mul(d2, splat<V>(0.5f)));
    const V ratio = mul(rr, mul(mul(isp, isp), isp));
    V l1 = fma(add(sp, sp), cos_third_acos(ratio), q);               // cos(theta / 3), theta = acos(ratio) in [0, pi]
    l1 = zip(l1, q, [](float a_, float b_) { return fmaxf(a_, b_); }); // l1 >= trace/3 always
    const V is1 = map(l1, [](float t) { return rsqrt_fast(t); });
    const V s1 = mul(l1, is1);
    const V inv1 = mul(is1, is1);
    // deflation: (s2 + S s3)^2 = (c1 - d^2/l1)/l1 + 2 d / s1
    const V w2 = fma(add(d, d), is1, mul(fma(neg(d2), inv1, c1), inv1));
    const V w = map(w2, [](float t) { return sqrt_fast(fmaxf(t, 0.0f)); });
    const V E0 = add(s1, w);

    // one Newton step on the quartic; skipped where f' is tiny against E^3 (s2 + S s3 -> 0: the
    // quartic's roots pair up and the deflated value above is the well-conditioned one)
    const V t = fma(E0, E0, neg(c2));
    const V d8 = mul(d, splat<V>(-8.0f));
    const V f = fma(t, t, fma(d8, E0, mul(c1, splat<V>(-4.0f))));
    const V fp = fma(mul(E0, splat<V>(4.0f)), t, d8);
    const V lim = mul(mul(E0, splat<V>(1e-3f)), mul(E0, E0));
    // M == 0 (L = 1, or every atom on the centroid): the floor above gives E0 ~ 3e-8 in units where |M| <= 2^8, i.e. below
    // 1e-5 A^2 in c^2 and clamped away where both models are points; a NaN in M gives q = NaN and passes through as NaN
    EPairT<V> r;
    r.E0 = E0;
    r.delta = zip3(f, fp, lim, [](float f_, float fp_, float lim_) { return fp_ > lim_ ? f_ * rcp_fast(fp_) : 0.0f; });
    return r;
}

template <class V>
__device__ __forceinline__ EPairT<V> eq2_energy(const V m[9])
{
    return eq2_energy(eq2_invariants(m));
}

// ---- FP64 form of the closed form for a pair (i, j) whose models carry power-of-two scales 2^ei, 2^ej:  m[] holds the
// Gram sums of the SCALED coordinates, S the sums of squares of the scaled coordinates, so
//   L c^2 2^-(ei+ej) = S_i 2^(ei-ej) + S_j 2^(ej-ei) - 2 E   with every scaling exact.   (The CUDA-core engine, which serves the long chains whose R_g^2 -- and with it
// every fp32 error term of the form above -- is largest).  Same mathematics: invariants of M, Viete's largest root and
// the deflated start value in fp32 (only a starting value), then Newton steps on the quartic in FP64 and the last
// line of eq. 2 in FP64, so that the result carries the rounding of the Gram sums and nothing else.
__device__ __forceinline__ float eq2_crmsd_f64(const double m[9], double S_i, int ei, double S_j, int ej, double invL)
{
    double c2 = 0.0;
#pragma unroll
    for (int i = 0; i < 9; ++i) c2 = fma(m[i], m[i], c2);
    double C[9];
    C[0] = m[4] * m[8] - m[5] * m[7];
    C[1] = m[5] * m[6] - m[3] * m[8];
    C[2] = m[3] * m[7] - m[4] * m[6];
    C[3] = m[7] * m[2] - m[8] * m[1];
    C[4] = m[8] * m[0] - m[6] * m[2];
    C[5] = m[6] * m[1] - m[7] * m[0];
    C[6] = m[1] * m[5] - m[2] * m[4];
    C[7] = m[2] * m[3] - m[0] * m[5];
    C[8] = m[0] * m[4] - m[1] * m[3];
    double c1 = 0.0;
#pragma unroll
    for (int i = 0; i < 9; ++i) c1 = fma(C[i], C[i], c1);
    const double d = m[0] * C[0] + m[1] * C[1] + m[2] * C[2];
    // starting value: the fp32 closed form on the rounded invariants, rescaled into the fp32 range by a power of two
    int e2 = 0;
    (void)frexp(c2, &e2);
    const int h = e2 / 2;                                             // c2 2^-2h in [0.25, 2)
    EqInvariants<float> inv;
    inv.c2 = (float)ldexp(c2, -2 * h);
    inv.c1 = (float)ldexp(c1, -4 * h);
    inv.d = (float)ldexp(d, -3 * h);
    const EPair e0 = eq2_energy(inv);
    double E = ldexp((double)e0.E0 - (double)e0.delta, h);
    if (c2 > 0.0) {
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const double t = fma(E, E, -c2);
            const double f = fma(t, t, -8.0 * d * E - 4.0 * c1);
            const double fp = 4.0 * E * t - 8.0 * d;
            if (fp > 1e-6 * E * E * E) E -= f / fp;                   // s2 + S s3 -> 0: keep the deflated value
        }
    } else {
        E = c2;                                                       // M == 0 -> 0; NaN stays NaN
    }
    const int de = max(-300, min(300, ei - ej));
    double res = (ldexp(S_i, de) - E) + (ldexp(S_j, -de) - E);
    res = res < 0.0 ? 0.0 : res;                                      // clamp (NaN stays NaN)
    return (float)sqrt(ldexp(res * invL, ei + ej));
}

// The same last line when each model carries T = sum |a|^2 in its TRUE scale as two floats (Thi, Tlo) and
// pw = 2^e (|e| <= 30, so every product below stays far inside the fp32 range):  with pp = pw_i pw_j,
//   L c^2 = (T_i - E pp) + (T_j - E pp);   E0 pp is exact, and each difference is exact by Sterbenz when the
// models are similar.  c = sqrt(max(0, .) / L) by the MUFU square root (relative error 2^-22 << 1e-3 A).
template <class V>
__device__ __forceinline__ V eq2_finish(const EPairT<V> e, V Thi_i, V Tlo_i, V pw_i, V Thi_j, V Tlo_j, V pw_j, float invL)
{
    using namespace lp;
    const V pp = mul(pw_i, pw_j);
    const V E0p = mul(e.E0, pp);
    const V res = add(add(sub(Thi_i, E0p), sub(Thi_j, E0p)), fma(mul(splat<V>(2.0f), e.delta), pp, add(Tlo_i, Tlo_j)));
    const V sc = mul(res, splat<V>(invL));
    return map(sc, [](float t) { return sqrt_fast(t < 0.0f ? 0.0f : t); });      // clamp (NaN stays NaN)
}

}  // namespace clusco
