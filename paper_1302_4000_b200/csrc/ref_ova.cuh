// ref_ova.cuh -- dRMSD (eq. 5) and contact map overlap (eq. 6-7) of N models against
// ONE reference structure ("... or with respect to the reference model").
//
// One warp per model, a single pass over the K = L(L-1)/2 atom pairs with both distances recomputed on the fly in FP64
// from coordinates held in shared memory (the reference once per CTA, one model per warp).  Unlike the all-versus-all
// forms there is no Gram identity here and no cancellation: dRMSD sums (d^A - d^B)^2 directly, CMO counts contacts.
// The work is O(N L^2) FP64 operations against O(N L) bytes, so the kernel is ALU-bound, not HBM-bound.
//   MODE 0: out[n] = sqrt( sum_{i<j} (d_ij^ref - d_ij^n)^2 / K )
//   MODE 1: out[n] = 100 * 2 n(ref and model) / (n(ref) + n(model)), contacts decided exactly as in drmsd_i8tc.cuh
//           (s < s_star, bit-identical to sqrt(s) < cutoff in FP64); two empty maps give 100.
#pragma once
#include "common.cuh"
#include "prep.cuh"

namespace clusco {

constexpr int ROVA_WARPS = 4;
constexpr int ROVA_MAX_L = 1024;

template <int MODE>
__global__ void __launch_bounds__(ROVA_WARPS * 32) ref_one_vs_all_kernel(const float* __restrict__ ref,
                                                                         const float* __restrict__ coords, int64_t N, int32_t L,
                                                                         double cutoff, float* __restrict__ out)
{
    extern __shared__ __align__(16) double rova_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* A = rova_smem;                                        // reference, 3 L doubles
    double* B = rova_smem + (size_t)(1 + warp) * 3 * L;           // this warp's model
    for (int e = threadIdx.x; e < 3 * L; e += blockDim.x) A[e] = (double)ref[e];
    __syncthreads();
    const int64_t K = (int64_t)L * (L - 1) / 2;
    // CMO: sqrt(s) < cutoff  <=>  s < s_star (see drmsd_prep_kernel)
    double s_star = 0.0;
    if (MODE == 1) {
        s_star = __dmul_rn(cutoff, cutoff);
        for (int it = 0; it < 8 && s_star > 0.0 && sqrt(s_star) >= cutoff; ++it) s_star = nextafter(s_star, 0.0);
        for (int it = 0; it < 8 && sqrt(s_star) < cutoff; ++it) s_star = nextafter(s_star, 1.0e300);
    }
    auto dist2 = [](const double* x, int i, int j) {
        const double dx = x[3 * i] - x[3 * j], dy = x[3 * i + 1] - x[3 * j + 1], dz = x[3 * i + 2] - x[3 * j + 2];
        return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    };
    for (int64_t n = (int64_t)blockIdx.x * ROVA_WARPS + warp; n < N; n += (int64_t)gridDim.x * ROVA_WARPS) {
        const float* x = coords + n * (int64_t)L * 3;
        bool finite = true;
        __syncwarp();
        for (int e = lane; e < 3 * L; e += 32) {
            const float v = x[e];
            finite = finite && fabsf(v) <= 3.0e38f;
            B[e] = (double)v;
        }
        finite = __all_sync(0xffffffffu, finite);
        __syncwarp();
        double sum = 0.0;
        int na = 0, nb = 0, nab = 0;
        int i = 0, pos = lane;                                   // entry k = lane, lane + 32, ...: pair (i, i + 1 + pos)
        for (int64_t k = lane; k < K; k += 32) {
            while (pos >= L - 1 - i) { pos -= L - 1 - i; ++i; }
            const int j = i + 1 + pos;
            const double sa = dist2(A, i, j), sb = dist2(B, i, j);
            if (MODE == 0) {
                const double diff = sqrt(sa) - sqrt(sb);
                sum += diff * diff;
            } else {
                const int ca = sa < s_star, cb = sb < s_star;
                na += ca; nb += cb; nab += ca & cb;
            }
            pos += 32;
        }
        if (MODE == 0) {
            sum = warp_sum(sum);
            if (lane == 0) out[n] = finite ? (float)sqrt(K > 0 ? sum / (double)K : 0.0) : __int_as_float(0x7fc00000);
        } else {
            na = __reduce_add_sync(0xffffffffu, na);
            nb = __reduce_add_sync(0xffffffffu, nb);
            nab = __reduce_add_sync(0xffffffffu, nab);
            if (lane == 0) {
                const double den = (double)na + (double)nb;
                const double S = den > 0.0 ? __ddiv_rn(__dmul_rn(200.0, (double)nab), den) : 100.0;
                out[n] = finite ? (float)S : __int_as_float(0x7fc00000);
            }
        }
    }
}

template <int MODE>
static inline int ref_one_vs_all_launch(const float* ref, const float* coords, int64_t N, int32_t L, double cutoff, float* out,
                                        int sms, cudaStream_t s)
{
    const size_t smem = (size_t)(1 + ROVA_WARPS) * 3 * (size_t)L * sizeof(double);
    CLUSCO_CUDA_TRY(cudaFuncSetAttribute(ref_one_vs_all_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1;
    CLUSCO_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ref_one_vs_all_kernel<MODE>, ROVA_WARPS * 32, smem));
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (N + ROVA_WARPS - 1) / ROVA_WARPS;
    const int64_t cap = (int64_t)sms * per_sm;
    if (grid > cap) grid = cap;
    ref_one_vs_all_kernel<MODE><<<(unsigned)grid, ROVA_WARPS * 32, smem, s>>>(ref, coords, N, L, cutoff, out);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

}  // namespace clusco
