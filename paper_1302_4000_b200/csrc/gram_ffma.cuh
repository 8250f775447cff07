// gram_ffma.cuh -- CUDA-core engine of the all-pairs kernel: steps a3 (covariance), a4 (eq. 2 closed form)
// and a5 (packed store) fused, one CTA per 32x32 tile of model pairs of the upper triangle.
//
// The nine sums of a pair are one 3x3 block of the product Y Y^T, Y = [3N x L] ("3x3
// covariance matrix M" -- here for all pairs at once).  Each thread owns 2x2 pairs = a 6x6 register
// block.  Accumulation is blocked: 16 atoms are summed into a fresh fp32 block, which is then added to
// an FP64 running total, so no fp32 chain is longer than 16 terms; the closed form runs in FP64
// (eq2_crmsd_f64).  This engine serves the chains too long for the tensor-core engine -- the most extended
// inputs, whose R_g^2 every fp32 error term scales with -- so it spends its spare issue slots on accuracy
// (DESIGN.md "Error budget").
#pragma once
#include "common.cuh"
#include "epilogue.cuh"

namespace clusco {

constexpr int FF_TILE = 32;          // models per tile side
constexpr int FF_KC = 16;            // atoms per shared-memory stage
constexpr int FF_LD = 3 * FF_TILE;   // floats per smem row (96)

struct TileRange {
    int64_t T;          // tile rows/cols in the whole matrix
    int64_t I_lo, I_hi; // tile-row range of this call
};

// linear tile index t (row-major over the upper triangle restricted to rows [I_lo, I_hi)) -> (I, J)
__device__ __forceinline__ void tile_from_linear(int64_t t, int64_t T, int64_t I_lo, int64_t& I, int64_t& J)
{
    // rows before row r (r = I - I_lo) hold r*W - r(r-1)/2 tiles, W = T - I_lo
    const double W = (double)(T - I_lo);
    double r = floor(((2.0 * W + 1.0) - sqrt((2.0 * W + 1.0) * (2.0 * W + 1.0) - 8.0 * (double)t)) * 0.5);
    int64_t ri = (int64_t)r;
    if (ri < 0) ri = 0;
    const int64_t Wi = T - I_lo;
    while (ri > 0 && ri * Wi - ri * (ri - 1) / 2 > t) --ri;
    while ((ri + 1) * Wi - (ri + 1) * ri / 2 <= t) ++ri;
    const int64_t before = ri * Wi - ri * (ri - 1) / 2;
    I = I_lo + ri;
    J = I + (t - before);
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <int MODE>
__global__ void __launch_bounds__(256, 2)
gram_ffma_kernel(const float* __restrict__ Yt, const ModelStat* __restrict__ stats, int64_t N, int64_t Np,
                 int32_t Lp16, float invL, TileRange tr, int64_t row_begin, int64_t row_end,
                 float* __restrict__ out, const Sink sink)
{
    __shared__ __align__(16) float As[2][FF_KC][FF_LD];
    __shared__ __align__(16) float Bs[2][FF_KC][FF_LD];

    int64_t I, J;
    tile_from_linear((int64_t)blockIdx.x, tr.T, tr.I_lo, I, J);
    const int64_t i_base = I * FF_TILE, j_base = J * FF_TILE;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int rp = 4 * (warp >> 1) + (lane >> 3);       // row pair 0..15
    const int cp = 8 * (warp & 1) + (lane & 7);         // col pair 0..15
    const int64_t ld = 3 * Np;

    auto load_stage = [&](int buf, int k0) {
#pragma unroll
        for (int it = 0; it < 3; ++it) {
            const int t = tid + 256 * it;                // 0..767 : [A|B][16 rows][24 float4]
            const int ab = t / 384, rem = t - 384 * ab;
            const int row = rem / 24, c4 = rem - 24 * row;
            const float* g = Yt + (int64_t)(k0 + row) * ld + 3 * (ab ? j_base : i_base) + 4 * c4;
            float* s = ab ? &Bs[buf][row][4 * c4] : &As[buf][row][4 * c4];
            cp_async16(s, g);
        }
        cp_async_commit();
    };

    double tot[36];
#pragma unroll
    for (int i = 0; i < 36; ++i) tot[i] = 0.0;

    const int nchunks = Lp16 / FF_KC;
    load_stage(0, 0);
    for (int c = 0; c < nchunks; ++c) {
        const int buf = c & 1;
        if (c + 1 < nchunks) {
            load_stage(buf ^ 1, (c + 1) * FF_KC);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        float acc[36];
#pragma unroll
        for (int i = 0; i < 36; ++i) acc[i] = 0.0f;
#pragma unroll
        for (int k = 0; k < FF_KC; ++k) {
            float a[6], b[6];
            const float2* ap = reinterpret_cast<const float2*>(&As[buf][k][6 * rp]);
            const float2* bp = reinterpret_cast<const float2*>(&Bs[buf][k][6 * cp]);
#pragma unroll
            for (int v = 0; v < 3; ++v) {
                const float2 av = ap[v], bv = bp[v];
                a[2 * v] = av.x; a[2 * v + 1] = av.y;
                b[2 * v] = bv.x; b[2 * v + 1] = bv.y;
            }
#pragma unroll
            for (int r = 0; r < 6; ++r)
#pragma unroll
                for (int s = 0; s < 6; ++s) acc[6 * r + s] = fmaf(a[r], b[s], acc[6 * r + s]);
        }
#pragma unroll
        for (int i = 0; i < 36; ++i) tot[i] += (double)acc[i];
        __syncthreads();
    }

    // ---- fused epilogue: eq. 2 per pair, packed store --------------------------------------------
    const int64_t base = packed_index(row_begin, row_begin + 1, N);
#pragma unroll
    for (int a = 0; a < 2; ++a) {
        const int64_t i = i_base + 2 * rp + a;
        if (i >= N || i < row_begin || i >= row_end) continue;
        const ModelStat si = stats[i];
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const int64_t j = j_base + 2 * cp + b;
            if (j >= N || j <= i) continue;
            const ModelStat sj = stats[j];
            double m[9];
#pragma unroll
            for (int p = 0; p < 3; ++p)
#pragma unroll
                for (int q = 0; q < 3; ++q) m[3 * p + q] = tot[6 * (3 * a + p) + 3 * b + q];
            const float c = eq2_crmsd_f64(m, (double)si.Shi + (double)si.Slo, si.ex, (double)sj.Shi + (double)sj.Slo,
                                          sj.ex, (double)invL);
            if (MODE == SINK_STORE) out[packed_index(i, j, N) - base] = c;
            else sink_emit<MODE>(sink, (int32_t)i, (int32_t)j, c);
        }
    }
}

}  // namespace clusco
