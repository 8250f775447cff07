// one_vs_all.cuh -- step a6: one reference structure against N models, a single
// HBM-bound pass over coords[N][L][3].
//
// `one_vs_all_stream_kernel` (L <= OVA_STREAM_MAX_L): every warp owns a private ring of shared-memory stages
// that one lane fills with 1-D bulk async copies (4 consecutive models = 48 L bytes per stage, 16-byte aligned
// by construction), so the global->shared path costs no load instructions and stays several stages deep.
// A stage is consumed by the whole warp, 8 lanes per model, in ONE pass of packed fp32 arithmetic (FFMA2): the
// coordinates are shifted by a point near the centroid (mean of four atoms), then the nine covariance sums
// against the centred native (shared memory, pre-expanded operand pairs), the coordinate sums and the sum of
// squares accumulate together -- sum_k a_k (x_k - ref) = sum_k a_k b_k because the native is centred, and the
// sum of squares about the centroid follows from the shifted moments.  Three butterfly steps reduce over the 8
// lanes; after 8 stages every lane owns the sums of ONE of 32 consecutive models, runs the eq. 2 closed form
// (epilogue.cuh) and the warp writes 32 consecutive results.
// `one_vs_all_kernel` is the plain-load variant kept for very long chains (one stage would not fit).
#pragma once
#include "common.cuh"
#include "epilogue.cuh"
#include "prep.cuh"
#include "tc_ptx.cuh"

namespace clusco {

// Sum of squares of the centred native as two floats.
struct NativeStat { float Shi, Slo; };

// Every CTA centres the native itself (FP64 centroid, a1 of the hot path for the reference structure) straight
// into its shared memory -- no scratch buffer, no extra launch; all CTAs of a launch get identical values
// because the reduction order depends on blockDim only.  EXPANDED = false: nat_s[k] = float4 (x, y, z, 0);
// EXPANDED = true: per 4-atom block and component p the twelve floats [a0 a0 a1 a1] [a2 a2 a3 a3] [a0 a1 a2 a3]
// (the FFMA2 operand pairs of ova_block), zero padded to 4 ceil(L/4) atoms.  Ends with a __syncthreads().
template <bool EXPANDED>
__device__ __forceinline__ NativeStat ova_native_to_smem(const float* __restrict__ native, int32_t L, float* nat_s)
{
    __shared__ double red[4][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
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
    double mean[3];
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        double v = 0.0;
        for (int w = 0; w < nw; ++w) v += red[p][w];
        mean[p] = v / (double)L;
    }
    double ss = 0.0;
    const int Lp = EXPANDED ? ((L + 3) & ~3) : L;
    for (int k = threadIdx.x; k < Lp; k += blockDim.x) {
        float a[3] = {0.0f, 0.0f, 0.0f};
        if (k < L) {
#pragma unroll
            for (int p = 0; p < 3; ++p) {
                a[p] = (float)((double)native[3 * k + p] - mean[p]);
                ss += (double)a[p] * a[p];
            }
        }
        if (EXPANDED) {
            float* q = nat_s + (k >> 2) * 36;
            const int i = k & 3;
#pragma unroll
            for (int p = 0; p < 3; ++p) {
                q[12 * p + 2 * i] = a[p];
                q[12 * p + 2 * i + 1] = a[p];
                q[12 * p + 8 + i] = a[p];
            }
        } else {
            reinterpret_cast<float4*>(nat_s)[k] = make_float4(a[0], a[1], a[2], 0.0f);
        }
    }
    ss = warp_sum(ss);
    if (lane == 0) red[3][warp] = ss;
    __syncthreads();
    double v = 0.0;
    for (int w = 0; w < nw; ++w) v += red[3][w];
    NativeStat r;
    r.Shi = (float)v;
    r.Slo = (float)(v - (double)r.Shi);
    return r;
}

// eq. 2 for one model from its ten sums (nine covariance sums against the centred native + sum of squares):
// scale M by an exact power of two so the cubic's coefficients stay in range, then
//   L c^2 2^-ex = S_native 2^-ex + S_model 2^-ex - 2 E
__device__ __forceinline__ float ova_finish(const float mine[10], float nShi, float nSlo, float invL)
{
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
    float res = (fmaf(nShi, sc, -e.E0) + fmaf(mine[9], sc, -e.E0)) + fmaf(2.0f, e.delta, nSlo * sc);
    res = res < 0.0f ? 0.0f : res;
    return sqrtf(res * invL * pow2i(ex - ex / 2) * pow2i(ex / 2));
}

// ---- streaming kernel ------------------------------------------------------------------------------------
constexpr int OVA_MPC = 4;                 // models per stage (one warp iteration), 8 lanes each
constexpr int OVA_MAX_WARPS = 16;
constexpr int OVA_STREAM_MAX_L = 2048;     // 2 stages of 48 L bytes + the native must fit in shared memory
constexpr int OVA_NATQ_FLOATS = 36;        // expanded native block, see ova_native_to_smem

// Six float2 = twelve consecutive floats (4 atoms: x0 y0 | z0 x1 | y1 z1 | x2 y2 | z2 x3 | y3 z3) of a staged
// model; VEC = widest aligned vector (floats) every model base and block offset allows: 4 if L % 4 == 0,
// 2 if L even, else 1
template <int VEC>
__device__ __forceinline__ void ova_load12(const float* p, float2 P[6])
{
    if (VEC == 4) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const float4 t = reinterpret_cast<const float4*>(p)[i];
            P[2 * i] = make_float2(t.x, t.y);
            P[2 * i + 1] = make_float2(t.z, t.w);
        }
    } else if (VEC == 2) {
#pragma unroll
        for (int i = 0; i < 6; ++i) P[i] = reinterpret_cast<const float2*>(p)[i];
    } else {
#pragma unroll
        for (int i = 0; i < 6; ++i) P[i] = make_float2(p[2 * i], p[2 * i + 1]);
    }
}

__device__ __forceinline__ float group8_sum(float v)
{
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    return v;
}

// running sums of one lane over its 4-atom blocks of one model, in the packed (two floats per register pair,
// FFMA2 / FADD2) form the xyz-interleaved input suggests: with B0..B5 the six shifted coordinate pairs of a
// block, native component p of atoms (0,0) (0,1) (1,1) multiplies (B0, B1, B2) and of atoms (2,2) (2,3) (3,3)
// multiplies (B3, B4, B5), so that  A[p] = (G_px, G_py),  B[p] = (G_pz, G_px),  C[p] = (G_py, G_pz).
struct OvaAcc {
    float2 SA, SB, SC;            // sums of the shifted coordinates: (x,y) (z,x) (y,z)
    float2 A[3], B[3], C[3];
    float2 Q0, Q1;                // sums of squares
};

__device__ __forceinline__ void ova_block(OvaAcc& acc, const float2 Bv[6], const float* __restrict__ nq)
{
    acc.SA = __fadd2_rn(acc.SA, __fadd2_rn(Bv[0], Bv[3]));
    acc.SB = __fadd2_rn(acc.SB, __fadd2_rn(Bv[1], Bv[4]));
    acc.SC = __fadd2_rn(acc.SC, __fadd2_rn(Bv[2], Bv[5]));
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const float4 n0 = reinterpret_cast<const float4*>(nq)[3 * p];        // a0 a0 a1 a1
        const float4 n1 = reinterpret_cast<const float4*>(nq)[3 * p + 1];    // a2 a2 a3 a3
        const float4 n2 = reinterpret_cast<const float4*>(nq)[3 * p + 2];    // a0 a1 a2 a3
        acc.A[p] = __ffma2_rn(make_float2(n0.x, n0.y), Bv[0], acc.A[p]);
        acc.B[p] = __ffma2_rn(make_float2(n2.x, n2.y), Bv[1], acc.B[p]);
        acc.C[p] = __ffma2_rn(make_float2(n0.z, n0.w), Bv[2], acc.C[p]);
        acc.A[p] = __ffma2_rn(make_float2(n1.x, n1.y), Bv[3], acc.A[p]);
        acc.B[p] = __ffma2_rn(make_float2(n2.z, n2.w), Bv[4], acc.B[p]);
        acc.C[p] = __ffma2_rn(make_float2(n1.z, n1.w), Bv[5], acc.C[p]);
    }
    acc.Q0 = __ffma2_rn(Bv[0], Bv[0], acc.Q0);
    acc.Q1 = __ffma2_rn(Bv[1], Bv[1], acc.Q1);
    acc.Q0 = __ffma2_rn(Bv[2], Bv[2], acc.Q0);
    acc.Q1 = __ffma2_rn(Bv[3], Bv[3], acc.Q1);
    acc.Q0 = __ffma2_rn(Bv[4], Bv[4], acc.Q0);
    acc.Q1 = __ffma2_rn(Bv[5], Bv[5], acc.Q1);
}

template <int VEC>
__global__ void __launch_bounds__(OVA_MAX_WARPS * 32, 1)
one_vs_all_stream_kernel(const float* __restrict__ native, const float* __restrict__ coords, int64_t N, int32_t L, float invL, int32_t stages,
                         float* __restrict__ out)
{
    extern __shared__ __align__(128) uint8_t ova_smem[];
    const int nblk = (L + 3) >> 2;                                  // 4-atom blocks per model
    const int nwarps = blockDim.x >> 5;
    const uint32_t stage_bytes = 48u * (uint32_t)L;
    float* nat_s = reinterpret_cast<float*>(ova_smem);              // nblk x 36 floats
    uint8_t* ring0 = ova_smem + (size_t)nblk * (OVA_NATQ_FLOATS * 4);
    uint64_t* bars0 = reinterpret_cast<uint64_t*>(ring0 + (size_t)nwarps * stages * stage_bytes);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0)
        for (int s = 0; s < stages; ++s) ptx::mbar_init(ptx::smem_u32(bars0 + warp * stages + s), 1);
    ptx::fence_mbar_init();
    const NativeStat nst = ova_native_to_smem<true>(native, L, nat_s);
    const float nShi = nst.Shi, nSlo = nst.Slo;

    uint8_t* ring = ring0 + (size_t)warp * stages * stage_bytes;
    const uint32_t bar = ptx::smem_u32(bars0 + warp * stages);
    const int64_t warp_g = (int64_t)blockIdx.x * nwarps + warp, n_warps = (int64_t)gridDim.x * nwarps;
    const int64_t n_batches = (N + 31) / 32;                        // a batch = 32 consecutive models = 8 stages
    const int64_t my_batches = warp_g < n_batches ? (n_batches - warp_g + n_warps - 1) / n_warps : 0;
    const uint32_t q_total = (uint32_t)(my_batches * 8);
    const int g = lane >> 3, s8 = lane & 7;

    // fill stage `st` with the 4 models of the warp's stage number q (warp-uniform)
    auto produce = [&](uint32_t q, uint32_t st) {
        const int64_t m0 = (warp_g + (int64_t)(q >> 3) * n_warps) * 32 + (q & 7) * OVA_MPC;
        const int64_t left = N - m0;
        const int cnt = left >= OVA_MPC ? OVA_MPC : (left > 0 ? (int)left : 0);
        const uint32_t bytes = (uint32_t)cnt * 12u * (uint32_t)L;
        uint8_t* dst = ring + (size_t)st * stage_bytes;
        if (cnt > 0 && (bytes & 15u) == 0) {
            if (lane == 0) {
                ptx::mbar_expect_tx(bar + 8u * st, bytes);
                ptx::bulk_g2s(ptx::smem_u32(dst), coords + m0 * (int64_t)L * 3, bytes, bar + 8u * st);
            }
        } else {
            // ragged last group whose byte count is not a multiple of 16: plain loads
            const float* src = coords + m0 * (int64_t)L * 3;
            for (int e = lane; e < cnt * 3 * L; e += 32) reinterpret_cast<float*>(dst)[e] = src[e];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar + 8u * st);
        }
    };

    for (uint32_t q = 0; q < (uint32_t)stages && q < q_total; ++q) produce(q, q);

    float mine[10];
#pragma unroll
    for (int v = 0; v < 10; ++v) mine[v] = 0.0f;
    // every lane walks blocks s8, s8 + 8, ...: n_uni iterations in which all eight lanes hold a full block, then
    // at most one ragged iteration (missing atoms are selected away)
    const int n_uni = (L >> 2) >> 3;
    const bool ragged = nblk > 8 * n_uni;
    const int c_last = 8 * n_uni + s8;
    const int natoms_last = max(0, min(4, L - 4 * c_last));
    const int c_last_eff = min(c_last, nblk - 1);
    // reference point of the single pass: the mean of four atoms spread along the chain
    const int r1 = L >> 2, r2 = L >> 1, r3 = (3 * L) >> 2;

    uint32_t st = 0, phase = 0;
    for (uint32_t q = 0; q < q_total; ++q) {
        ptx::mbar_wait(bar + 8u * st, phase);
        const float* xs = reinterpret_cast<const float*>(ring + (size_t)st * stage_bytes) + (size_t)g * 3 * L;
        // shift by a point near the centroid: sum_k a_k (x_k - ref) = sum_k a_k b_k because the native is centred,
        // and sum |x - ref|^2 - L |mean - ref|^2 = sum |b|^2 loses nothing when |mean - ref| < R_g
        const float rx = 0.25f * ((xs[0] + xs[3 * r1]) + (xs[3 * r2] + xs[3 * r3]));
        const float ry = 0.25f * ((xs[1] + xs[3 * r1 + 1]) + (xs[3 * r2 + 1] + xs[3 * r3 + 1]));
        const float rz = 0.25f * ((xs[2] + xs[3 * r1 + 2]) + (xs[3 * r2 + 2] + xs[3 * r3 + 2]));
        const float2 nXY = make_float2(-rx, -ry), nZX = make_float2(-rz, -rx), nYZ = make_float2(-ry, -rz);
        OvaAcc acc;
        acc.SA = acc.SB = acc.SC = acc.Q0 = acc.Q1 = make_float2(0.f, 0.f);
#pragma unroll
        for (int p = 0; p < 3; ++p) acc.A[p] = acc.B[p] = acc.C[p] = make_float2(0.f, 0.f);
        const float* pm = xs + 12 * s8;
        const float* pn = nat_s + OVA_NATQ_FLOATS * s8;
#pragma unroll 2
        for (int it = 0; it < n_uni; ++it) {
            float2 P[6];
            ova_load12<VEC>(pm, P);
            P[0] = __fadd2_rn(P[0], nXY); P[1] = __fadd2_rn(P[1], nZX); P[2] = __fadd2_rn(P[2], nYZ);
            P[3] = __fadd2_rn(P[3], nXY); P[4] = __fadd2_rn(P[4], nZX); P[5] = __fadd2_rn(P[5], nYZ);
            ova_block(acc, P, pn);
            pm += 96;
            pn += 8 * OVA_NATQ_FLOATS;
        }
        if (ragged) {
            float2 P[6];
            ova_load12<VEC>(xs + 12 * c_last_eff, P);
            const bool w0 = natoms_last > 0, w1 = natoms_last > 1, w2 = natoms_last > 2, w3 = natoms_last > 3;
            P[0] = make_float2(w0 ? P[0].x - rx : 0.f, w0 ? P[0].y - ry : 0.f);
            P[1] = make_float2(w0 ? P[1].x - rz : 0.f, w1 ? P[1].y - rx : 0.f);
            P[2] = make_float2(w1 ? P[2].x - ry : 0.f, w1 ? P[2].y - rz : 0.f);
            P[3] = make_float2(w2 ? P[3].x - rx : 0.f, w2 ? P[3].y - ry : 0.f);
            P[4] = make_float2(w2 ? P[4].x - rz : 0.f, w3 ? P[4].y - rx : 0.f);
            P[5] = make_float2(w3 ? P[5].x - ry : 0.f, w3 ? P[5].y - rz : 0.f);
            ova_block(acc, P, nat_s + OVA_NATQ_FLOATS * c_last_eff);
        }
        // the stage is consumed: refill it, then reduce while the copy flies
        __syncwarp();
        if (q + stages < q_total) produce(q + stages, st);
        float G[10];
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            G[3 * p] = group8_sum(acc.A[p].x + acc.B[p].y);
            G[3 * p + 1] = group8_sum(acc.A[p].y + acc.C[p].x);
            G[3 * p + 2] = group8_sum(acc.B[p].x + acc.C[p].y);
        }
        const float sx = group8_sum(acc.SA.x + acc.SB.y), sy = group8_sum(acc.SA.y + acc.SC.x),
                    sz = group8_sum(acc.SB.x + acc.SC.y);
        const float qq = group8_sum((acc.Q0.x + acc.Q0.y) + (acc.Q1.x + acc.Q1.y));
        // sum |b|^2 = sum |x - ref|^2 - |sum (x - ref)|^2 / L
        G[9] = fmaf(-invL, fmaf(sx, sx, fmaf(sy, sy, sz * sz)), qq);
        const bool keep = s8 == (int)(q & 7);
#pragma unroll
        for (int v = 0; v < 10; ++v)
            if (keep) mine[v] = G[v];
        if ((q & 7) == 7) {
            // lane (g, s8) holds model 4 s8 + g of the batch: the warp writes 32 consecutive floats
            const int64_t m = (warp_g + (int64_t)(q >> 3) * n_warps) * 32 + 4 * s8 + g;
            if (m < N) out[m] = ova_finish(mine, nShi, nSlo, invL);
        }
        if (++st == (uint32_t)stages) { st = 0; phase ^= 1; }
    }
}

static inline size_t ova_stream_smem(int32_t L, int warps, int stages)
{
    return (size_t)((L + 3) / 4) * (OVA_NATQ_FLOATS * 4) + (size_t)warps * stages * 48 * (size_t)L + (size_t)warps * stages * 8;
}
// warps per CTA and stages per warp for chains of L atoms: up to 12 warps with 2 stages each, then as many more
// stages as it takes to keep ~96 KB of bulk copies in flight per SM (short chains have small stages)
static inline bool ova_stream_config(int32_t L, int* warps, int* stages)
{
    if (L > OVA_STREAM_MAX_L) return false;
    const size_t budget = 226 * 1024;                    // 227 KB per CTA minus the static reduction scratch
    int w = 12;
    while (w > 1 && ova_stream_smem(L, w, 2) > budget) --w;
    if (ova_stream_smem(L, w, 2) > budget) return false;
    const size_t per_stage = (size_t)w * 48 * (size_t)L;
    int st = 1 + (int)((96 * 1024 + per_stage - 1) / per_stage);
    if (st > 8) st = 8;
    while (st > 2 && ova_stream_smem(L, w, st) > budget) --st;
    *warps = w;
    *stages = st;
    return true;
}

constexpr int OVA_WARPS = 8;

__global__ void __launch_bounds__(OVA_WARPS * 32)
one_vs_all_kernel(const float* __restrict__ native, const float* __restrict__ coords, int64_t N, int32_t L, float invL, float* __restrict__ out)
{
    extern __shared__ float4 nat_s[];                     // centred native, L float4
    const NativeStat nst = ova_native_to_smem<false>(native, L, reinterpret_cast<float*>(nat_s));
    const float nShi = nst.Shi, nSlo = nst.Slo;

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
        if (lane < cnt) out[m0 + lane] = ova_finish(mine, nShi, nSlo, invL);
    }
}

}  // namespace clusco
