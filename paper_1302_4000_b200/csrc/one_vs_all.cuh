// one_vs_all.cuh -- step a6: one reference structure against N models, a single
// HBM-bound pass.  Each warp owns blocks of 32 consecutive models: for every model the 32 lanes stride
// over its atoms (centroid, then the nine covariance sums against the centred native and the sum of
// squares), warp-reduce, and lane t keeps model t's sums; after 32 models all lanes run the eq. 2
// closed form (epilogue.cuh) in parallel and write 32 consecutive results.
#pragma once
#include "common.cuh"
#include "epilogue.cuh"
#include "prep.cuh"

namespace clusco {

// Native: centred in FP64, stored as float4 (x, y, z, 0); sum of squares as two floats.
struct NativeStat { float Shi, Slo; };

// one CTA; writes natc[L] (float4) and nstat
__global__ void __launch_bounds__(256) native_prep_kernel(const float* __restrict__ native, int32_t L,
                                                          float4* __restrict__ natc, NativeStat* __restrict__ nstat)
{
    __shared__ double red[3][8];
    __shared__ double mean[3];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double s[3] = {0.0, 0.0, 0.0};
    for (int k = threadIdx.x; k < L; k += blockDim.x) {
        s[0] += (double)native[3 * k];
        s[1] += (double)native[3 * k + 1];
        s[2] += (double)native[3 * k + 2];
    }
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const double v = warp_sum(s[p]);
        if (lane == 0) red[p][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = 0.0;
        for (int w = 0; w < 8; ++w) v += red[threadIdx.x][w];
        mean[threadIdx.x] = v / (double)L;
    }
    __syncthreads();
    double ss = 0.0;
    for (int k = threadIdx.x; k < L; k += blockDim.x) {
        const float ax = (float)((double)native[3 * k] - mean[0]);
        const float ay = (float)((double)native[3 * k + 1] - mean[1]);
        const float az = (float)((double)native[3 * k + 2] - mean[2]);
        natc[k] = make_float4(ax, ay, az, 0.0f);
        ss += (double)ax * ax + (double)ay * ay + (double)az * az;
    }
    ss = warp_sum(ss);
    __syncthreads();
    if (lane == 0) red[0][warp] = ss;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int w = 0; w < 8; ++w) v += red[0][w];
        nstat->Shi = (float)v;
        nstat->Slo = (float)(v - (double)nstat->Shi);
    }
}

constexpr int OVA_WARPS = 8;

__global__ void __launch_bounds__(OVA_WARPS * 32)
one_vs_all_kernel(const float4* __restrict__ natc, const NativeStat* __restrict__ nstat,
                  const float* __restrict__ coords, int64_t N, int32_t L, float invL, float* __restrict__ out)
{
    extern __shared__ float4 nat_s[];                     // centred native, L float4
    for (int k = threadIdx.x; k < L; k += blockDim.x) nat_s[k] = natc[k];
    __syncthreads();
    const float nShi = nstat->Shi, nSlo = nstat->Slo;

    const int lane = threadIdx.x & 31;
    const int64_t warp_g = (int64_t)blockIdx.x * OVA_WARPS + (threadIdx.x >> 5);
    const int64_t n_warps = (int64_t)gridDim.x * OVA_WARPS;
    const int64_t n_blocks = (N + 31) / 32;

    for (int64_t blk = warp_g; blk < n_blocks; blk += n_warps) {
        float mine[10];
#pragma unroll
        for (int v = 0; v < 10; ++v) mine[v] = 0.0f;
        const int64_t m0 = blk * 32;
        const int cnt = (int)min((int64_t)32, N - m0);
        for (int t = 0; t < cnt; ++t) {
            const float* x = coords + (m0 + t) * (int64_t)L * 3;
            // centroid
            float sx = 0.f, sy = 0.f, sz = 0.f;
            for (int k = lane; k < L; k += 32) {
                sx += x[3 * k];
                sy += x[3 * k + 1];
                sz += x[3 * k + 2];
            }
            const float mx = warp_sum(sx) * invL, my = warp_sum(sy) * invL, mz = warp_sum(sz) * invL;
            // covariance sums (native centred => sum_k n_k = 0) and sum of squares
            float g[10];
#pragma unroll
            for (int v = 0; v < 10; ++v) g[v] = 0.0f;
            for (int k = lane; k < L; k += 32) {
                const float bx = x[3 * k] - mx, by = x[3 * k + 1] - my, bz = x[3 * k + 2] - mz;
                const float4 a = nat_s[k];
                g[0] = fmaf(a.x, bx, g[0]); g[1] = fmaf(a.x, by, g[1]); g[2] = fmaf(a.x, bz, g[2]);
                g[3] = fmaf(a.y, bx, g[3]); g[4] = fmaf(a.y, by, g[4]); g[5] = fmaf(a.y, bz, g[5]);
                g[6] = fmaf(a.z, bx, g[6]); g[7] = fmaf(a.z, by, g[7]); g[8] = fmaf(a.z, bz, g[8]);
                g[9] = fmaf(bx, bx, fmaf(by, by, fmaf(bz, bz, g[9])));
            }
#pragma unroll
            for (int v = 0; v < 10; ++v) {
                const float s = warp_sum(g[v]);
                if (lane == t) mine[v] = s;
            }
        }
        if (lane < cnt) {
            // scale M by an exact power of two so the cubic's coefficients stay in range
            float gmax = 0.0f;
#pragma unroll
            for (int v = 0; v < 9; ++v) gmax = fmaxf(gmax, fabsf(mine[v]));
            int ex = 0;
            if (gmax > 0.0f && gmax < 3.0e38f) (void)frexpf(gmax, &ex);
            ex = max(-100, min(100, ex));
            const float sc = pow2i(-ex);
            float m[9];
#pragma unroll
            for (int v = 0; v < 9; ++v) m[v] = mine[v] * sc;
            const EPair e = eq2_energy(m);
            // L c^2 2^-ex = S_native 2^-ex + S_model 2^-ex - 2 E
            float res = (fmaf(nShi, sc, -e.E0) + fmaf(mine[9], sc, -e.E0)) + fmaf(2.0f, e.delta, nSlo * sc);
            res = res < 0.0f ? 0.0f : res;
            out[m0 + lane] = sqrtf(res * invL * pow2i(ex - ex / 2) * pow2i(ex / 2));
        }
    }
}

}  // namespace clusco
