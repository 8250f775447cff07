// prep.cuh -- steps a1 + a2 of the hot path: centring and sum of squares per model (implicit in eq. 2:
// M and the radius of gyration are taken about the centroid), plus the re-layout of the
// centred coordinates into the operand planes the Gram engines read.
#pragma once
#include "common.cuh"

namespace clusco {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// ---- stats: one warp per model ---------------------------------------------------------------------
// mean (FP64), exponent ex with max|a| * 2^-ex in [0.5, 1), S = sum (a 2^-ex)^2 as two floats.
// Models n >= N (padding up to Np) get a neutral record.
__global__ void __launch_bounds__(256) model_stats_kernel(const float* __restrict__ coords, int64_t N,
                                                          int64_t Np, int32_t L, ModelStat* __restrict__ stats)
{
    const int lane = threadIdx.x & 31;
    const int64_t n = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (n >= Np) return;
    if (n >= N) {
        if (lane == 0) {
            ModelStat s;
            s.mean[0] = s.mean[1] = s.mean[2] = 0.0;
            s.Shi = s.Slo = 0.0f;
            s.ex = 0;
            s.pad = 0;
            stats[n] = s;
        }
        return;
    }
    const float* x = coords + n * (int64_t)L * 3;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int k = lane; k < L; k += 32) {
        sx += (double)x[3 * k];
        sy += (double)x[3 * k + 1];
        sz += (double)x[3 * k + 2];
    }
    const double invL = 1.0 / (double)L;
    const double mx = warp_sum(sx) * invL, my = warp_sum(sy) * invL, mz = warp_sum(sz) * invL;
    double ss = 0.0;
    float amax = 0.0f;
    for (int k = lane; k < L; k += 32) {
        const float ax = (float)((double)x[3 * k] - mx);
        const float ay = (float)((double)x[3 * k + 1] - my);
        const float az = (float)((double)x[3 * k + 2] - mz);
        amax = fmaxf(amax, fmaxf(fabsf(ax), fmaxf(fabsf(ay), fabsf(az))));
        ss += (double)ax * ax + (double)ay * ay + (double)az * az;
    }
    ss = warp_sum(ss);
    amax = warp_max(amax);
    if (lane == 0) {
        int ex = 0;
        if (amax > 0.0f && amax < 3.0e38f) (void)frexpf(amax, &ex);      // amax = m 2^ex, m in [0.5,1)
        ex = max(-100, min(100, ex));
        const double S = ldexp(ss, -2 * ex);                             // exact rescale
        ModelStat s;
        s.mean[0] = mx; s.mean[1] = my; s.mean[2] = mz;
        s.Shi = (float)S;
        s.Slo = (float)(S - (double)s.Shi);
        s.ex = ex;
        s.pad = 0;
        stats[n] = s;
    }
}

// ---- FFMA operand plane: Yt[k][3 n + p] = a_{n,k,p} 2^-ex_n, fp32, zero padded ---------------------
// grid (Np/32, ceil(Lp16/64)); block 256.  Coalesced read of 32 models x 64 atoms, transposed through
// shared memory, written as rows of 96 contiguous floats.
__global__ void __launch_bounds__(256) ffma_plane_kernel(const float* __restrict__ coords, int64_t N,
                                                         int64_t Np, int32_t L, int32_t Lp16,
                                                         const ModelStat* __restrict__ stats,
                                                         float* __restrict__ Yt)
{
    __shared__ float tile[64][100];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t n0 = (int64_t)blockIdx.x * 32;
    const int k0 = blockIdx.y * 64;
    for (int mi = warp; mi < 32; mi += 8) {
        const int64_t n = n0 + mi;
        double dmean[3] = {0., 0., 0.};
        float sc = 0.0f;
        if (n < N) {
            dmean[0] = stats[n].mean[0]; dmean[1] = stats[n].mean[1]; dmean[2] = stats[n].mean[2];
            sc = pow2i(-stats[n].ex);
        }
        const float* x = coords + n * (int64_t)L * 3;
        for (int e = lane; e < 192; e += 32) {
            const int ka = e / 3, p = e - 3 * ka;
            const int k = k0 + ka;
            float v = 0.0f;
            if (n < N && k < L)
                v = (float)((double)x[3 * k + p] - (p == 0 ? dmean[0] : (p == 1 ? dmean[1] : dmean[2]))) * sc;
            tile[ka][3 * mi + p] = v;
        }
    }
    __syncthreads();
    const int64_t ld = 3 * Np;
    for (int t = threadIdx.x; t < 64 * 24; t += 256) {
        const int ka = t / 24, c4 = t - 24 * ka;
        const int k = k0 + ka;
        if (k < Lp16) {
            const float4 v = make_float4(tile[ka][4 * c4], tile[ka][4 * c4 + 1], tile[ka][4 * c4 + 2],
                                         tile[ka][4 * c4 + 3]);
            *reinterpret_cast<float4*>(Yt + (int64_t)k * ld + 3 * n0 + 4 * c4) = v;
        }
    }
}

// ---- public clusco_center: centred[N][L][3] and r2[N] (steps a1 + a2 on their own) -----------------
// One warp per model, ONE pass over HBM: the model's 3 L floats are read once -- as 16-byte vectors over the aligned
// interior of its range in the flat coordinate array, scalars at the ragged ends (a model starts at float 3 L n, which is
// 16-byte aligned only for every fourth n in general) -- into a warp-private shared-memory strip, with the three FP64
// coordinate sums taken on the way (component = position mod 3); the centred values and the FP64 sum of squares come from
// the strip, and the output leaves by the same aligned-vector / ragged-scalar scheme.  Bound: HBM, 24 N L + 4 N bytes.
constexpr int CENTER_WARPS = 4;
constexpr int CENTER_MAX_FLOATS = 12 * 1024;       // strip capacity per warp (48 KB): L <= 4096; longer chains take center_long_kernel

__global__ void __launch_bounds__(CENTER_WARPS * 32) center_kernel(const float* coords, int64_t N, int32_t L, int32_t strip_floats,
                                                                  float* centred, float* __restrict__ r2)
{
    extern __shared__ __align__(16) float center_strip[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t n = (int64_t)blockIdx.x * CENTER_WARPS + wib;
    if (n >= N) return;
    const int n_el = 3 * L;
    const int64_t e0 = n * (int64_t)n_el;                  // first float of the model in the flat array
    const int head = (int)((4 - (e0 & 3)) & 3);            // floats before the first 16-byte boundary
    const int lead = head < n_el ? head : n_el;
    const int nvec = (n_el - lead) >> 2;
    // strip position = lead-relative: strip[4 + (e - lead)] for e >= lead, strip[4 - lead + e] for the head, so that the
    // vector part of the strip is 16-byte aligned too
    float* strip = center_strip + (size_t)wib * strip_floats + 4 - lead;
    const float* x = coords + e0;
    // vector part: lane handles vectors lane, lane + 32, ...; float e = lead + 4 v + i has component (lead + 4 v + i) % 3
    double sv[3] = {0.0, 0.0, 0.0};
    // (four vectors per lane are requested before the first is used: 2 KB in flight per warp)
    for (int v0 = lane; v0 < nvec; v0 += 128) {
        float4 t[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (v0 + 32 * u < nvec) t[u] = *reinterpret_cast<const float4*>(x + lead + 4 * (v0 + 32 * u));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int v = v0 + 32 * u;
            if (v < nvec) {
                *reinterpret_cast<float4*>(strip + lead + 4 * v) = t[u];
                const int c = (lead + 4 * v) % 3;          // component of .x; .y, .z, .w follow cyclically
                const double a = (double)t[u].x + (double)t[u].w, b = (double)t[u].y, d = (double)t[u].z;
                // components (c, c+1, c+2, c) -> add into the per-component sums
                if (c == 0) { sv[0] += a; sv[1] += b; sv[2] += d; }
                else if (c == 1) { sv[1] += a; sv[2] += b; sv[0] += d; }
                else { sv[2] += a; sv[0] += b; sv[1] += d; }
            }
        }
    }
    // ragged ends: the head (< 4 floats) and the tail after the last whole vector (< 4 floats)
    const int tail0 = lead + 4 * nvec;
    for (int e = lane; e < lead + (n_el - tail0); e += 32) {
        const int ee = e < lead ? e : tail0 + (e - lead);
        const float t = x[ee];
        strip[ee] = t;
        sv[ee % 3] += (double)t;
    }
    const double invL = 1.0 / (double)L;
    const double m0 = warp_sum(sv[0]) * invL, m1 = warp_sum(sv[1]) * invL, m2 = warp_sum(sv[2]) * invL;
    __syncwarp();
    double ss = 0.0;
    float* y = centred ? centred + e0 : nullptr;
    for (int v = lane; v < nvec; v += 32) {
        const float4 t = *reinterpret_cast<const float4*>(strip + lead + 4 * v);
        const int c = (lead + 4 * v) % 3;
        const double mc0 = c == 0 ? m0 : (c == 1 ? m1 : m2), mc1 = c == 0 ? m1 : (c == 1 ? m2 : m0),
                     mc2 = c == 0 ? m2 : (c == 1 ? m0 : m1);
        const double a0 = (double)t.x - mc0, a1 = (double)t.y - mc1, a2 = (double)t.z - mc2, a3 = (double)t.w - mc0;
        ss += a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3;
        if (y) *reinterpret_cast<float4*>(y + lead + 4 * v) = make_float4((float)a0, (float)a1, (float)a2, (float)a3);
    }
    for (int e = lane; e < lead + (n_el - tail0); e += 32) {
        const int ee = e < lead ? e : tail0 + (e - lead);
        const int c = ee % 3;
        const double a = (double)strip[ee] - (c == 0 ? m0 : (c == 1 ? m1 : m2));
        ss += a * a;
        if (y) y[ee] = (float)a;
    }
    ss = warp_sum(ss);
    if (r2 && lane == 0) r2[n] = (float)(ss * invL);
}

// chains too long for the strip: two passes over the model (the second one mostly from L2)
__global__ void __launch_bounds__(256) center_long_kernel(const float* coords, int64_t N, int32_t L,
                                                          float* centred, float* __restrict__ r2)
{
    const int lane = threadIdx.x & 31;
    const int64_t n = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (n >= N) return;
    const float* x = coords + n * (int64_t)L * 3;
    double s[3] = {0.0, 0.0, 0.0};
    for (int e = lane; e < 3 * L; e += 32) s[e % 3] += (double)x[e];
    const double invL = 1.0 / (double)L;
    const double m0 = warp_sum(s[0]) * invL, m1 = warp_sum(s[1]) * invL, m2 = warp_sum(s[2]) * invL;
    double ss = 0.0;
    float* y = centred ? centred + n * (int64_t)L * 3 : nullptr;
    for (int e = lane; e < 3 * L; e += 32) {
        const int p = e % 3;
        const double a = (double)x[e] - (p == 0 ? m0 : (p == 1 ? m1 : m2));
        ss += a * a;
        if (y) y[e] = (float)a;
    }
    ss = warp_sum(ss);
    if (r2 && lane == 0) r2[n] = (float)(ss * invL);
}

}  // namespace clusco
