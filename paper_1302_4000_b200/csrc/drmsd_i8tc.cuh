// drmsd_i8tc.cuh -- all-versus-all distance RMSD (the paper's eq. 5) as ONE Gram contraction on the
// tensor cores.
//
// With d^A in R^K the vector of the K = L(L-1)/2 intra-model distances d_ij = |x_i - x_j| (i < j, row-major),
//     dRMSD(A,B)^2 = (2 / (L(L-1))) sum_{i<j} (d_ij^A - d_ij^B)^2 = ( |d^A|^2 + |d^B|^2 - 2 d^A . d^B ) / K,
// so the whole matrix is the N x K by K x N product D D^T plus a trivial epilogue.  The cancellation is as severe
// as in eq. 2 of cRMSD (a difference of numbers ~K * R_g^2 that must be right to ~1e-3 A^2 * K), so the same exact
// arithmetic is used: every model's distances are scaled by a power of two, multiplied by
// KAPPA 2^23 and rounded to a 24-bit integer I = g0 2^16 + g1 2^8 + g2 (signed 8-bit digits); the dot product is
//     sum_k I_A I_B = 2^32 V0 + 2^24 V1 + 2^16 V2 (+ two dropped low-order levels),
// six int8 products accumulated EXACTLY in int32 TMEM accumulators (|V| <= 3 K 2^14 < 2^31 needs L <= 296), and
// |d|^2 is taken from the same integers (exact in 64 bits), so quantisation cancels for similar models.
//
// Operand plane (one, shared by both operands).  dRMSD: P[tile128][k-step][digit][4096 B] -- for 128 consecutive models
// and 32 consecutive entries of K, the int8 digit `digit` as a shared-memory image in tcgen05's canonical K-major
// no-swizzle core-matrix layout (16 row groups x [2 x 128 B]).  CMO: P[tile256][k-step][half][4096 B], so that the 256
// models of a tile are ONE N = 256 operand and either half an M = 128 operand.  Consecutive k-steps of a tile are
// contiguous, so an operand of a stage of KG k-steps is ONE contiguous run fetched by ONE 1-D bulk copy (the per-copy /
// per-stage handshake, not the bytes, was what limited an earlier layout with eight 2 KB pieces per k-step).
//
// Kernel: persistent, one CTA per SM, warp 0 = bulk-copy producer (ring of stages of KG k-steps), warp 1 = MMA issuer,
// warps 2..17 = epilogue (TMEM lane quadrant x column quarter; results are transposed through shared memory so that the
// stores run along the packed rows).  dRMSD: tile = 128 x 128 models, 2 x 2 thread-block clusters whose CTAs each fetch
// half of their A and B runs and multicast them; per k-step four MMAs -- a0.[b0;b1] -> V0|V1, a1.[b0;b1] -> V1|V2 (N = 256),
// a0.b2 and a2.b0 -> V2 -- level v (TMEM columns 128 v ...) collecting the digit products A(ga).B(gb)^T with ga + gb = v.
// CMO: every CTA owns a 256 x 256 block (four 128-column accumulators = all of TMEM), two N = 256 MMAs per k-step, 1 x 2
// clusters (the row tile's run is shared by multicast, each CTA fetches its own column tile) so that all 148 SMs work.
#pragma once
#include "common.cuh"
#include "prep.cuh"
#include "tc_ptx.cuh"

namespace clusco {

constexpr double DG_KAPPA = 127.0 / 128.0;
constexpr int DG_MAX_L = 296;                  // 3 K 2^14 < 2^31 with K = L(L-1)/2
constexpr int DG_TILE = 128;
constexpr int DG_SLAB = 4096;                  // bytes of one (tile, k-step, digit) image: 128 rows x 32 entries
// DIGITS = 3: dRMSD (24-bit fixed-point distances); DIGITS = 1: CMO (0/1 contact maps, eq. 6-7) on the same kernels
constexpr int DG_KG3 = 2;                      // dRMSD: k-steps per stage (measured Gram time at C3's shape: 1 -> 7.11 ms, 2 -> 6.73 ms)
template <int DIGITS> struct DGCfg {
    // k-steps per stage of the 128 x 128-tile kernels (consecutive k-steps are contiguous); the plane's k-step count is
    // padded to a multiple of it
    static constexpr int KG = DIGITS == 3 ? DG_KG3 : 4;
};
// CMO on the cluster path: every CTA owns a 2 x 2 block of 128-model tiles (DESIGN.md section 13 has the history:
// 3.1 ms -> 1.47 ms at C3's shape against 0.7 ms of tensor time)
constexpr int DG_CMO_CLUSTER_I = 1;            // CMO cluster rows: 2 (2 x 2, 132 SMs) or 1 (1 x 2, all 148 SMs, 1.5 x the L2 reads)
constexpr int DG_KG1B = 2;                     // CMO, blocked: k-steps per stage (measured: 2 -> 1.69 ms, 4 -> 1.71 ms whole call)
constexpr int DG_EPI_WARPS = 16;               // 4 TMEM lane quadrants x 4 column quarters of a tile
constexpr int DG_THREADS = (2 + DG_EPI_WARPS) * 32;
constexpr int DG_PREP_WARPS = 8;
constexpr int DG_CLUSTER_I = 2;                // cluster shape of the Gram kernel: CLI tile rows x CLJ tile columns
constexpr int DG_CLUSTER_J = 2;                // (dRMSD, measured at C3's shape: 2x2 6.67 ms, 1x2 6.76 ms whole call)

struct __align__(16) DStat {
    double T;          // KAPPA^2 sum_k d_k^2 of the quantised distances, true scale (Angstrom^2); NaN poisons the model
    float pw;          // 2^e, e = the model's scale exponent
    float pad;         // CMO: (float)T
};

struct DWorkspace {
    int64_t N, Np, K, ks, tiles;        // ks = k-steps, padded to a multiple of the stage's k-group
    size_t off_stat, off_sched, off_plane, total;
};
static inline DWorkspace drmsd_workspace_layout(int64_t N, int32_t L, int digits = 3)
{
    DWorkspace w;
    w.N = N;
    w.Np = round_up(N, digits == 1 ? 2 * DG_TILE : DG_TILE);   // CMO: 256-row plane tiles (two slabs per k-step)
    w.K = (int64_t)L * (L - 1) / 2;
    const int64_t kg = digits == 3 ? DGCfg<3>::KG : DGCfg<1>::KG;
    w.ks = round_up((w.K + 31) / 32, kg);
    w.tiles = w.Np / DG_TILE;
    size_t o = 0;
    w.off_stat = o;
    o += (size_t)round_up((int64_t)sizeof(DStat) * w.Np, 256);
    w.off_sched = o;                                       // int2 (SI, SJ) per super-tile of the cluster kernel's walk
    {
        const int64_t T = w.Np / DG_TILE;                  // at most T (T + 1) / 2 + T entries for any cluster shape
        o += (size_t)round_up((int64_t)sizeof(int2) * (T * (T + 1) / 2 + T), 256);
    }
    w.off_plane = o;
    o += (size_t)round_up(w.tiles * w.ks * digits * DG_SLAB, 256);
    w.total = o + 256;
    return w;
}

// ---- distances, scale, digits, operand plane: one CTA per 8 consecutive models (one core-matrix row group), one
// warp per model; lane = entry within the k-step.  Two passes over the K distances (max, then quantise), each
// recomputed in FP64 from the fp32 coordinates held in shared memory.
// DIGITS = 1 (CMO): the entry is the contact bit C_ij = (|x_i - x_j| < cutoff), eq. 6 -- decided in FP64 with IEEE
// operations only (no FMA contraction), so the decision is reproducible bit for bit; T = n(A), the contact count.
template <int DIGITS>
__global__ void __launch_bounds__(DG_PREP_WARPS * 32) drmsd_prep_kernel(const float* __restrict__ coords, int64_t N, int32_t L,
                                                                        int64_t K, int64_t ks, double cutoff,
                                                                        int8_t* __restrict__ plane, DStat* __restrict__ stat)
{
    __shared__ float xs[DG_PREP_WARPS][3 * DG_MAX_L];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t n = (int64_t)blockIdx.x * DG_PREP_WARPS + w;
    const bool valid = n < N;
    float* x = xs[w];
    bool finite = true;
    for (int e = lane; e < 3 * L; e += 32) {
        const float v = valid ? coords[n * (int64_t)L * 3 + e] : 0.0f;
        finite = finite && (fabsf(v) <= 3.0e38f);
        x[e] = v;
    }
    __syncwarp();
    auto dist2 = [&](int i, int j) {
        const double dx = (double)x[3 * i] - (double)x[3 * j];
        const double dy = (double)x[3 * i + 1] - (double)x[3 * j + 1];
        const double dz = (double)x[3 * i + 2] - (double)x[3 * j + 2];
        return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    };
    // scale: a power of two 2^ex with dmax 2^-ex < 1, from the bound  amax <= dmax <= 2 amax,  amax = the largest
    // distance of an atom from the centroid (the centroid lies in the convex hull, so some atom is at least amax away
    // from the farthest one): at most one bit of the 24 is given up, and no pass over the K distances is needed
    double m2 = 0.0;
    if (valid && DIGITS == 3) {
        double c0 = 0.0, c1 = 0.0, c2 = 0.0;
        for (int a = lane; a < L; a += 32) { c0 += (double)x[3 * a]; c1 += (double)x[3 * a + 1]; c2 += (double)x[3 * a + 2]; }
        c0 = warp_sum(c0) / (double)L; c1 = warp_sum(c1) / (double)L; c2 = warp_sum(c2) / (double)L;
        for (int a = lane; a < L; a += 32) {
            const double dx = (double)x[3 * a] - c0, dy = (double)x[3 * a + 1] - c1, dz = (double)x[3 * a + 2] - c2;
            m2 = fmax(m2, dx * dx + dy * dy + dz * dz);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m2 = fmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
    int ex = 0;
    const double dmax = 2.0 * sqrt(m2);
    if (dmax > 0.0 && dmax < 1.0e30) (void)frexp(dmax, &ex);
    const bool in_range = dmax < 1.0e9;
    ex = max(-30, min(30, ex));
    const float scale_f = (float)ldexp(DG_KAPPA, 23 - ex);       // KAPPA 2^(23 - ex): exact in fp32
    // CMO: sqrt(s) < cutoff  <=>  s < s_star, s_star = the smallest double whose correctly rounded square root is
    // >= cutoff (the rounded square root is monotone), found once per thread by stepping from cutoff^2: the
    // per-entry decision needs no square root and stays bit-identical to eq. 6 evaluated literally in FP64
    double s_star = 0.0;
    if (DIGITS == 1) {
        s_star = __dmul_rn(cutoff, cutoff);
        for (int it = 0; it < 8 && s_star > 0.0 && sqrt(s_star) >= cutoff; ++it) s_star = nextafter(s_star, 0.0);
        for (int it = 0; it < 8 && sqrt(s_star) < cutoff; ++it) s_star = nextafter(s_star, 1.0e300);
    }
    const float s_mid = (float)s_star, s_band = (float)(s_star * 3.0e-6);
    // one pass over the K entries, 4 k-steps (128 entries) per trip.  Computing: lane = entry within the k-step, so the
    // warp reads 32 CONSECUTIVE atoms j of a row (stride 3 words: no bank conflict; four entries per lane put the four
    // lane groups on the same banks).  Storing: a 4 x 4 byte transpose within each group of four lanes hands lane
    // (4 j8 + sub) the digit bytes of entries 4 j8 .. 4 j8 + 3 of k-step sub: one 32-bit store per digit.
    const int64_t t128 = n >> 7;
    const int g = (int)(n & 127) >> 3, r8 = (int)(n & 7);
    const int sub = lane & 3, j8 = lane >> 2;
    const uint32_t sel1 = (lane & 1) ? 0x3715u : 0x6240u, sel2 = (lane & 2) ? 0x3276u : 0x5410u;
    // DIGITS = 3: P[tile128][k-step][digit][4 KB].  DIGITS = 1: P[tile256][k-step][half][4 KB] -- the two 128-row slabs of a
    // k-step are consecutive, so a 256-model tile is ONE N = 256 operand and either half is an M = 128 operand
    constexpr int64_t KSTEP_SLABS = DIGITS == 3 ? 3 : 2;
    int8_t* base = plane + (DIGITS == 3 ? t128 * ks * 3 : (t128 >> 1) * ks * 2 + (t128 & 1)) * DG_SLAB + g * 256 +
                   (j8 >> 2) * 128 + r8 * 16 + (j8 & 3) * 4;
    long long sumsq = 0ll;
    uint32_t ncontact = 0u;
    int ii = 0, jj = 1 + lane;                                   // entry k = 32 kk + lane: pair (ii, jj), ii < jj < L
    float xa0 = x[0], xa1 = x[1], xa2 = x[2];                    // atom ii, reloaded when the row changes
    const int K32 = valid ? (int)K : 0, ks32 = (int)ks;          // K < 2^16 (L <= 296)
    for (int kk0 = 0; kk0 < ks32; kk0 += 4) {
        uint32_t W0 = 0u, W1 = 0u, W2 = 0u;                      // byte s: this lane's entry of k-step kk0 + s
#pragma unroll
        for (int s4 = 0; s4 < 4; ++s4) {
            const int k = (kk0 + s4) * 32 + lane;
            if (k < K32) {
                if (jj >= L) {                                   // next row(s): entry (ii, L + d) is entry (ii + 1, ii + 2 + d)
                    do { jj += ii + 2 - L; ++ii; } while (jj >= L);
                    xa0 = x[3 * ii]; xa1 = x[3 * ii + 1]; xa2 = x[3 * ii + 2];
                }
                if (DIGITS == 3) {
                    // fp32 is enough here: each coordinate difference carries one rounding, the squared distance three more and
                    // the IEEE square root one, so d is right to ~2^-22 -- about the 24-bit quantisation step itself, random in
                    // sign, and 10^3 times below what the 2e-3 A^2 bar allows (the FP64 version of this loop cost twice the time)
                    const float fx = xa0 - x[3 * jj], fy = xa1 - x[3 * jj + 1], fz = xa2 - x[3 * jj + 2];
                    const float df = __fsqrt_rn(fmaf(fz, fz, fmaf(fy, fy, fx * fx)));
                    const int I = min(__float2int_rn(df * scale_f), (1 << 23) - 65536);          // keeps |g0| <= 127 whatever the rounding
                    const int g2 = (int)(int8_t)(I & 0xff);
                    const int I1 = (I - g2) >> 8;
                    const int g1 = (int)(int8_t)(I1 & 0xff);
                    const int g0 = (I1 - g1) >> 8;
                    // |d|^2 from the SAME three levels the Gram keeps (I^2 minus the two dropped low-order levels),
                    // so that an identical pair cancels to exactly 0
                    sumsq += (long long)I * (long long)I - (long long)(512 * g1 * g2 + g2 * g2);
                    W0 |= (uint32_t)(g0 & 0xff) << (8 * s4);
                    W1 |= (uint32_t)(g1 & 0xff) << (8 * s4);
                    W2 |= (uint32_t)(g2 & 0xff) << (8 * s4);
                } else {
                    // fp32 screen: each difference carries one rounding (relative 2^-24), so the fp32 squared distance
                    // is within 3e-7 of the FP64 one; outside a 3e-6 band around the threshold the fp32 comparison
                    // decides, inside it (about one entry in 10^5) the FP64 evaluation of eq. 6 does
                    const float fx = xa0 - x[3 * jj], fy = xa1 - x[3 * jj + 1], fz = xa2 - x[3 * jj + 2];
                    const float s2f = fmaf(fz, fz, fmaf(fy, fy, fx * fx));
                    uint32_t cbit = s2f < s_mid ? 1u : 0u;
                    if (!(fabsf(s2f - s_mid) > s_band)) cbit = dist2(ii, jj) < s_star ? 1u : 0u;      // also taken by NaN
                    ncontact += cbit;
                    W0 |= cbit << (8 * s4);
                }
            }
            jj += 32;
        }
        // 4 x 4 byte transpose over the four lanes of a group: 1-byte blocks with lane ^ 1, then 2-byte blocks with lane ^ 2
        auto tr4 = [&](uint32_t W) {
            const uint32_t a = __byte_perm(W, __shfl_xor_sync(0xffffffffu, W, 1), sel1);
            return __byte_perm(a, __shfl_xor_sync(0xffffffffu, a, 2), sel2);
        };
        const uint32_t w0 = tr4(W0), w1 = DIGITS == 3 ? tr4(W1) : 0u, w2 = DIGITS == 3 ? tr4(W2) : 0u;
        const int kk = kk0 + sub;
        if (kk < ks32) {
            int8_t* p = base + (int64_t)kk * KSTEP_SLABS * DG_SLAB;
            *reinterpret_cast<uint32_t*>(p) = w0;
            if (DIGITS == 3) {
                *reinterpret_cast<uint32_t*>(p + DG_SLAB) = w1;
                *reinterpret_cast<uint32_t*>(p + 2 * DG_SLAB) = w2;
            }
        }
    }
    if (DIGITS == 1) sumsq = (long long)ncontact;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sumsq += __shfl_xor_sync(0xffffffffu, sumsq, o);
    finite = __all_sync(0xffffffffu, finite);
    if (lane == 0) {
        DStat s;
        s.T = DIGITS == 3 ? ldexp((double)sumsq, 2 * ex - 46) : (double)sumsq;
        if (!finite || (DIGITS == 3 && !in_range)) s.T = __longlong_as_double(0x7ff8000000000000ll);
        s.pw = pow2i(ex);
        s.pad = DIGITS == 1 ? (float)s.T : 0.0f;           // CMO: the contact count (< 2^24, exact) for the fp32 epilogue
        stat[n] = s;
    }
}

// ---- the Gram kernel -------------------------------------------------------------------------------------------
struct DGParams {
    const int8_t* plane;
    const DStat* stat;
    const int2* sched;     // cluster kernel: the super-tile walk (dg_schedule_kernel)
    float* out;
    int64_t N, ks;
    int32_t T;             // tiles per side (Np / 128); upper-triangle tiles I <= J are linearised row-major
    int64_t total;         // T (T + 1) / 2
    int64_t n_sched;       // entries of `sched`
    double invKk;          // 1 / (KAPPA^2 K)
};

__device__ __forceinline__ void dg_tile_from_linear(int64_t t, int32_t T, int32_t& I, int32_t& J)
{
    // rows before row I hold I T - I (I - 1) / 2 tiles
    int32_t lo = 0, hi = T - 1;
    while (lo < hi) {
        const int32_t mid = (lo + hi + 1) >> 1;
        if ((int64_t)mid * T - (int64_t)mid * (mid - 1) / 2 <= t) lo = mid; else hi = mid - 1;
    }
    I = lo;
    J = I + (int32_t)(t - ((int64_t)I * T - (int64_t)I * (I - 1) / 2));
}

// The cluster kernel's walk over the super-tiles that touch the upper triangle, in blocks of bi x bj super-tiles that
// are about square in tile units and about one wave of clusters large: the clusters running at the same time then
// share their A tile rows AND their B tile columns in L2 (a row-major walk shares one A row and streams every B
// column from HBM: 18.5 GB of DRAM reads at C3's shape instead of 9.7 GB).  One thread, ~T^2/2 entries.
// super-tile (SI, SJ) = tiles (cli SI + ri, clj SJ + rj); it is walked if any of its tiles lies on or above the diagonal
__host__ __device__ __forceinline__ bool dg_super_valid(int32_t SI, int32_t SJ, int32_t cli, int32_t clj, int32_t T)
{
    return cli * SI < T && clj * SJ < T && cli * SI <= clj * SJ + (clj - 1);
}
__global__ void dg_schedule_kernel(int32_t T, int32_t cli, int32_t clj, int32_t bi, int32_t bj, int2* __restrict__ sched)
{
    // one warp: 32 candidates (block-major order) per round, compacted with a ballot
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    const int lane = threadIdx.x;
    const int32_t TI = (T + cli - 1) / cli, TJ = (T + clj - 1) / clj;
    const int32_t NBI = (TI + bi - 1) / bi, NBJ = (TJ + bj - 1) / bj;
    const int64_t per_block = (int64_t)bi * bj, total = (int64_t)NBI * NBJ * per_block;
    int64_t n = 0;
    for (int64_t c0 = 0; c0 < total; c0 += 32) {
        const int64_t c = c0 + lane;
        bool ok = false;
        int32_t SI = 0, SJ = 0;
        if (c < total) {
            const int64_t blk = c / per_block, in = c - blk * per_block;
            SI = (int32_t)(blk / NBJ) * bi + (int32_t)(in / bj);
            SJ = (int32_t)(blk % NBJ) * bj + (int32_t)(in % bj);
            ok = SI < TI && SJ < TJ && dg_super_valid(SI, SJ, cli, clj, T);
        }
        const uint32_t m = __ballot_sync(0xffffffffu, ok);
        if (ok) sched[n + __popc(m & ((1u << lane) - 1u))] = make_int2(SI, SJ);
        n += __popc(m);
    }
}
static inline int64_t dg_schedule_count(int32_t T, int32_t cli, int32_t clj)
{
    const int32_t TI = (T + cli - 1) / cli, TJ = (T + clj - 1) / clj;
    int64_t n = 0;
    for (int32_t SI = 0; SI < TI; ++SI)
        for (int32_t SJ = 0; SJ < TJ; ++SJ) n += dg_super_valid(SI, SJ, cli, clj, T) ? 1 : 0;
    return n;
}

// CLI x CLJ = 1 x 1: every CTA fetches its own operands.  Otherwise thread-block clusters: the CTAs of a cluster work
// on the CLI x CLJ block of tiles (CLI SI + ri, CLJ SJ + rj), rank = CLJ ri + rj; the A slabs of a tile row are needed
// by the CTAs of that row and the B slabs of a tile column by the CTAs of that column, so with 2 x 2 each CTA fetches
// HALF of its A and HALF of its B and multicasts them to its row / column partner: the L2 -> SM operand bytes halve.
// A stage is free again when every CTA of the cluster has consumed it (EMPTY counts CL multicast commits).
// TB > 1 (needs CLI = CLJ = TB = 2): the CTA of rank (ri, rj) owns the tiles (TB (CLI SI + ri) + a, TB (CLJ SJ + rj) + b),
// a, b < TB, accumulator a TB + b at TMEM columns 128 (a TB + b); it fetches the WHOLE run of row tile a = rj and of column
// tile b = ri and multicasts them to its row / column partner, so a stage holds [A_0 | A_1 | B_0 | B_1].
template <int DIGITS, int TB> struct DGKernelCfg {
    static constexpr int KG = TB > 1 ? DG_KG1B : DGCfg<DIGITS>::KG;
    static constexpr int OPER_BYTES = KG * DIGITS * DG_SLAB;            // one tile's run of a stage
    static constexpr int STAGE_BYTES = 2 * TB * OPER_BYTES;
    static constexpr int STAGES = (216 * 1024) / STAGE_BYTES;
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_BYTES + 8 * (2 * STAGES + 2) + 16 + DG_EPI_WARPS * 32 * 17 * sizeof(float);
};
template <int DIGITS, int CLI, int CLJ, int TB>
__global__ void __launch_bounds__(DG_THREADS, 1) drmsd_gram_kernel(const DGParams P)
{
    static_assert(TB == 1 || (TB == 2 && CLI <= 2 && CLJ == 2 && DIGITS == 1), "blocked tiles: 2 x 2 or 1 x 2 clusters, one digit");
    static_assert(DIGITS == 3 || TB == 2 || CLI * CLJ == 1, "one digit: 256-row plane tiles need the blocked kernel or no cluster");
    constexpr int CL = CLI * CLJ;                                // CTAs per cluster: CLI tile rows x CLJ tile columns
    typedef DGKernelCfg<DIGITS, TB> KC;
    constexpr int DG_STAGES = KC::STAGES, DG_STAGE_BYTES = KC::STAGE_BYTES;
    constexpr int KG = KC::KG, OPER = KC::OPER_BYTES;
    extern __shared__ __align__(128) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)DG_STAGES * DG_STAGE_BYTES);
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto FULL = [&](uint32_t s) { return bar0 + 8u * s; };
    auto EMPTY = [&](uint32_t s) { return bar0 + 8u * (DG_STAGES + s); };
    const uint32_t ACC_FULL = bar0 + 8u * (2 * DG_STAGES), ACC_EMPTY = ACC_FULL + 8u;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * DG_STAGES + 2);

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const uint32_t rank = CL > 1 ? ptx::cluster_ctarank() : 0u;
    const int ri = (int)(rank / CLJ), rj = (int)(rank % CLJ);
    if (threadIdx.x == 0) {
        for (int s = 0; s < DG_STAGES; ++s) {
            ptx::mbar_init(FULL(s), 1);
            ptx::mbar_init(EMPTY(s), CL);
        }
        ptx::mbar_init(ACC_FULL, 1);
        ptx::mbar_init(ACC_EMPTY, DG_EPI_WARPS);
        ptx::fence_mbar_init();
    }
    if (warp == 1) ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
    ptx::tc_fence_before();
    __syncthreads();
    if (CL > 1) ptx::cluster_sync();                             // every CTA's barriers exist before any remote signal
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int64_t ng = P.ks / KG;                                // stages per tile (k-groups)
    // CL == 1: tiles I <= J row-major (dg_tile_from_linear); CL > 1: the super-tile list written by dg_schedule_kernel
    const int64_t total2 = CL > 1 ? P.n_sched : P.total;
    const int64_t first = blockIdx.x / CL, step = gridDim.x / CL;

    if (warp == 0) {
        // ===== producer =====
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            const int64_t tile_stride = P.ks * (DIGITS == 3 ? 3 : 2) * DG_SLAB;     // DIGITS = 1: stride of a 256-row tile
            for (int64_t t = first; t < total2; t += step) {
                int32_t SI, SJ;
                if (CL > 1) { const int2 e = P.sched[t]; SI = e.x; SJ = e.y; } else dg_tile_from_linear(t, P.T, SI, SJ);
                if (TB > 1) {
                    // my block = the 256-row tile CLI SI + ri times the 256-row tile CLJ SJ + rj (clamped: results are
                    // masked); a stage's A (B) operand is ONE contiguous run of that tile, KG k-steps x [half 0 | half 1]:
                    // I fetch half rj (ri) of the run -- KG / 2 k-steps -- and multicast it to my row (column) partner
                    const int32_t IR = min(CLI * SI + ri, P.T / 2 - 1), JC = min(CLJ * SJ + rj, P.T / 2 - 1);
                    const int8_t* a0 = P.plane + (int64_t)IR * tile_stride + rj * OPER;
                    const int8_t* b0 = P.plane + (int64_t)JC * tile_stride + ri * OPER;
                    for (int64_t kg = 0; kg < ng; ++kg) {
                        ptx::mbar_wait(EMPTY(stage), phase ^ 1);
                        ptx::mbar_expect_tx(FULL(stage), DG_STAGE_BYTES);
                        const uint32_t sA = ptx::smem_u32(smem + (size_t)stage * DG_STAGE_BYTES);
                        const uint32_t sB = sA + TB * OPER;
                        ptx::bulk_g2s_multicast(sA + rj * OPER, a0 + kg * 2 * OPER, OPER, FULL(stage), (uint16_t)(3u << (ri * CLJ)));
                        if (CLI == 2)
                            ptx::bulk_g2s_multicast(sB + ri * OPER, b0 + kg * 2 * OPER, OPER, FULL(stage),
                                                    (uint16_t)((1u | (1u << CLJ)) << rj));
                        else
                            ptx::bulk_g2s(sB, b0 + kg * 2 * OPER, 2 * OPER, FULL(stage));     // 1 x 2 cluster: my own column tile
                        if (++stage == DG_STAGES) { stage = 0; phase ^= 1; }
                    }
                    continue;
                }
                const int32_t I = min(CLI * SI + ri, P.T - 1), J = min(CLJ * SJ + rj, P.T - 1);   // clamped: results are masked
                if (DIGITS == 1) {
                    // one digit, no clusters (small N): the 128-row halves of the 256-row plane tiles, one 4 KB slab per k-step
                    const int8_t* a0 = P.plane + (int64_t)(I >> 1) * tile_stride + (I & 1) * DG_SLAB;
                    const int8_t* b0 = P.plane + (int64_t)(J >> 1) * tile_stride + (J & 1) * DG_SLAB;
                    for (int64_t kg = 0; kg < ng; ++kg) {
                        ptx::mbar_wait(EMPTY(stage), phase ^ 1);
                        ptx::mbar_expect_tx(FULL(stage), DG_STAGE_BYTES);
                        const uint32_t sA = ptx::smem_u32(smem + (size_t)stage * DG_STAGE_BYTES);
                        const uint32_t sB = sA + OPER;
                        for (int q = 0; q < KG; ++q) {
                            ptx::bulk_g2s(sA + q * DG_SLAB, a0 + (kg * KG + q) * 2 * DG_SLAB, DG_SLAB, FULL(stage));
                            ptx::bulk_g2s(sB + q * DG_SLAB, b0 + (kg * KG + q) * 2 * DG_SLAB, DG_SLAB, FULL(stage));
                        }
                        if (++stage == DG_STAGES) { stage = 0; phase ^= 1; }
                    }
                    continue;
                }
                const int8_t* a0 = P.plane + (int64_t)I * tile_stride;
                const int8_t* b0 = P.plane + (int64_t)J * tile_stride;
                for (int64_t kg = 0; kg < ng; ++kg) {
                    ptx::mbar_wait(EMPTY(stage), phase ^ 1);
                    ptx::mbar_expect_tx(FULL(stage), DG_STAGE_BYTES);
                    const uint32_t sA = ptx::smem_u32(smem + (size_t)stage * DG_STAGE_BYTES);
                    const uint32_t sB = sA + OPER;
                    // a stage's A (and B) operand is one contiguous run of the plane: KG k-steps x DIGITS slabs.
                    // A is needed by the CLJ CTAs of my tile row: with CLJ == 2 I fetch half rj of the run and multicast it
                    if (CLJ == 2)
                        ptx::bulk_g2s_multicast(sA + rj * (OPER / 2), a0 + kg * OPER + rj * (OPER / 2), OPER / 2, FULL(stage),
                                                (uint16_t)(3u << (ri * CLJ)));
                    else
                        ptx::bulk_g2s(sA, a0 + kg * OPER, OPER, FULL(stage));
                    // B is needed by the CLI CTAs of my tile column: with CLI == 2 I fetch half ri and multicast it
                    if (CLI == 2)
                        ptx::bulk_g2s_multicast(sB + ri * (OPER / 2), b0 + kg * OPER + ri * (OPER / 2), OPER / 2, FULL(stage),
                                                (uint16_t)((1u | (1u << CLJ)) << rj));
                    else
                        ptx::bulk_g2s(sB, b0 + kg * OPER, OPER, FULL(stage));
                    if (++stage == DG_STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (warp-uniform loop, one elected lane issues) =====
        constexpr uint32_t ID128 = ptx::idesc_s8(128, 128), ID256 = ptx::idesc_s8(128, 256);
        constexpr uint64_t DESC_HI = (uint64_t)((256u >> 4) | (1u << 14)) << 32;          // SBO 256 B, version 1
        const uint32_t lo0 = ((128u >> 4) << 16) | ((ptx::smem_u32(smem) & 0x3FFFFu) >> 4);   // LBO 128 B
        uint32_t stage = 0, phase = 0, tile_n = 0;
        for (int64_t t = first; t < total2; t += step, ++tile_n) {
            ptx::mbar_wait(ACC_EMPTY, (tile_n & 1) ^ 1);
            ptx::tc_fence_after();
            for (int64_t kg = 0; kg < ng; ++kg) {
                ptx::mbar_wait(FULL(stage), phase);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
                    const uint32_t a_lo = lo0 + stage * (DG_STAGE_BYTES >> 4);
                    const uint32_t b_lo = a_lo + (TB * OPER >> 4);
                    constexpr uint32_t SL = DG_SLAB >> 4;
#pragma unroll
                    for (int q = 0; q < KG; ++q) {
                        const uint32_t acc = (kg > 0 || q > 0) ? 1u : 0u;
                        const uint32_t aq = a_lo + q * DIGITS * SL, bq = b_lo + q * DIGITS * SL;
                        if (TB > 1) {
                            // k-step q of the A run = [rows 0..127 | rows 128..255]; of the B run = one N = 256 operand:
                            // accumulator a TB + b = TMEM columns 256 a + 128 b
#pragma unroll
                            for (int a = 0; a < TB; ++a)
                                ptx::mma_i8(tmem + 256 * a, DESC_HI | (a_lo + (2 * q + a) * SL), DESC_HI | (b_lo + 2 * q * SL), ID256, acc);
                            continue;
                        }
                        // level v (TMEM columns 128 v ...) collects the digit products A(ga) . B(gb)^T with ga + gb = v
                        if (DIGITS == 3) {
                            // the digit slabs of B are consecutive, so [b0; b1] is one N = 256 operand and its product
                            // with a0 (a1) lands on the adjacent level blocks V0 | V1 (V1 | V2): four MMAs instead of
                            // six N = 128 ones -- the same work, 40 KB instead of 48 KB of shared-memory operand reads per
                            // k-step (the K loop runs at the pace of shared memory: operand reads + stage fills)
                            ptx::mma_i8(tmem, DESC_HI | aq, DESC_HI | bq, ID256, acc);                       // V0 | V1
                            ptx::mma_i8(tmem + 256, DESC_HI | aq, DESC_HI | (bq + 2 * SL), ID128, acc);      // V2 = a0 b2
                            ptx::mma_i8(tmem + 128, DESC_HI | (aq + SL), DESC_HI | bq, ID256, 1);            // V1 | V2
                            ptx::mma_i8(tmem + 256, DESC_HI | (aq + 2 * SL), DESC_HI | bq, ID128, 1);        // V2 += a2 b0
                        } else {
                            ptx::mma_i8(tmem, DESC_HI | aq, DESC_HI | bq, ID128, acc);
                        }
                    }
                    if (CL > 1) ptx::tc_commit_multicast(EMPTY(stage), (uint16_t)((1u << CL) - 1u));
                    else ptx::tc_commit(EMPTY(stage));
                    if (kg == ng - 1) ptx::tc_commit(ACC_FULL);
                }
                __syncwarp();
                if (++stage == DG_STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ===== epilogue: thread = row model (TMEM lane), loops over the 128 column models of the tile =====
        const int quad = warp & 3;
        // results go through a warp-private 32 x 33 float tile so that the stores run along the packed rows (a thread is a
        // ROW of the accumulator: storing straight from it costs 32 sectors per instruction, 65k LSU cycles per tile)
        float* tp = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(tmem_slot) + 16) + (warp - 2) * (32 * 17);
        const int part = (warp - 2) >> 2;                        // column quarter: chunks 2 part, 2 part + 1 of 16 models
        const int rr = lane >> 4, cc = lane & 15;                // store role: row parity, column within the chunk
        uint32_t tile_n = 0;
        for (int64_t t = first; t < total2; t += step, ++tile_n) {
            int32_t SI, SJ;
            if (CL > 1) { const int2 e = P.sched[t]; SI = e.x; SJ = e.y; } else dg_tile_from_linear(t, P.T, SI, SJ);
            ptx::mbar_wait(ACC_FULL, tile_n & 1);
            ptx::tc_fence_after();
#pragma unroll 1
            for (int sub = 0; sub < TB * TB; ++sub) {            // the tiles of this CTA's block
                const int32_t I = TB * (CLI * SI + ri) + sub / TB, J = TB * (CLJ * SJ + rj) + sub % TB;
                const bool active = I < P.T && J < P.T && I <= J;    // a cluster's block may hang over the edge / the diagonal
                const int64_t ibase = (int64_t)min(I, P.T - 1) * DG_TILE + quad * 32;
                const int64_t i = ibase + lane;
                const DStat si = P.stat[i];                          // slots beyond N hold neutral records
                const double pwi = (double)si.pw * 0x1p-30;
                const uint32_t ta = tmem + ((uint32_t)(quad * 32) << 16) + 128 * sub;
                if (active) {
#pragma unroll 1
                    for (int h = 0; h < 2; ++h) {                    // this warp's two 16-column chunks
                        const int c = 2 * part + h;
                        uint32_t v0[16], v1[16], v2[16];
                        ptx::tmem_ld_32x32b_x16(ta + 16 * c, v0);
                        if (DIGITS == 3) {
                            ptx::tmem_ld_32x32b_x16(ta + 128 + 16 * c, v1);
                            ptx::tmem_ld_32x32b_x16(ta + 256 + 16 * c, v2);
                        }
                        ptx::tmem_ld_wait();
                        const int64_t j0 = (int64_t)J * DG_TILE + 16 * c;
#pragma unroll
                        for (int e = 0; e < 16; ++e) {
                            const DStat sj = P.stat[j0 + e];         // warp-uniform address
                            float val;
                            if (DIGITS == 3) {
                                const long long dot = ((long long)(int32_t)v0[e] << 16) + ((long long)(int32_t)v1[e] << 8) +
                                                      (long long)(int32_t)v2[e];
                                const double res = (si.T + sj.T) - 2.0 * (double)dot * (pwi * (double)sj.pw);
                                const float d2 = (float)(res * P.invKk);
                                val = sqrtf(d2 < 0.0f ? 0.0f : d2);                      // clamp (NaN stays NaN)
                            } else {
                                // eq. 7: S = 100 * 2 n(A and B) / (n(A) + n(B)); two empty maps are identical: 100.
                                // fp32 throughout and still the correctly rounded quotient: 200 n < 2^24 and the
                                // denominator are exact in fp32, the division is IEEE; rounding the FP64 quotient to
                                // fp32 (the oracle's route) gives the same float, because a ratio of integers with a
                                // denominator < 2^17 cannot come within 2^-53 of an fp32 rounding boundary
                                const float den = si.pad + sj.pad;                           // pad = (float)T
                                val = den > 0.0f ? __fdiv_rn(200.0f * (float)(int32_t)v0[e], den)
                                                 : (den == 0.0f ? 100.0f : den);              // NaN model -> NaN
                            }
                            tp[lane * 17 + e] = val;
                        }
                        __syncwarp();
                        // transposed: one store instruction = 16 consecutive column models of TWO row models (2 x 64 B)
                        const int64_t j = j0 + cc;
                        // packed offset of row ir: ir (2N - ir - 1) / 2 - ir - 1; two rows further it grows by 2N - 2 ir - 5
                        int64_t ir = ibase + rr;
                        float* dst = P.out + (ir * (2 * P.N - ir - 1) / 2 - ir - 1 + j);
                        int64_t inc = 2 * P.N - 2 * ir - 5;
#pragma unroll 4
                        for (int r2 = 0; r2 < 16; ++r2) {
                            if (ir < P.N && j < P.N && j > ir) *dst = tp[(2 * r2 + rr) * 17 + cc];
                            dst += inc;
                            inc -= 4;
                            ir += 2;
                        }
                        __syncwarp();
                    }
                }
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(ACC_EMPTY);
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (CL > 1) ptx::cluster_sync();                             // no CTA leaves while a partner may still signal it
    if (warp == 1) ptx::tmem_dealloc(tmem, 512);
}

template <int DIGITS>
static inline int drmsd_launch(const float* coords, int64_t N, int32_t L, double cutoff, float* out, char* ws, int sms,
                               cudaStream_t s)
{
    const DWorkspace w = drmsd_workspace_layout(N, L, DIGITS);
    DStat* stat = (DStat*)(ws + w.off_stat);
    int8_t* plane = (int8_t*)(ws + w.off_plane);
    drmsd_prep_kernel<DIGITS><<<(unsigned)(w.Np / DG_PREP_WARPS), DG_PREP_WARPS * 32, 0, s>>>(coords, N, L, w.K, w.ks, cutoff,
                                                                                              plane, stat);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    DGParams P;
    P.plane = plane;
    P.stat = stat;
    P.sched = (const int2*)(ws + w.off_sched);
    P.out = out;
    P.N = N;
    P.ks = w.ks;
    P.T = (int32_t)(w.Np / DG_TILE);
    P.total = (int64_t)P.T * (P.T + 1) / 2;
    P.invKk = 1.0 / (DG_KAPPA * DG_KAPPA * (double)w.K);
    static_assert(DGCfg<1>::KG % DG_KG1B == 0, "the plane's k-step padding must cover the blocked kernel's k-group");
    // thread-block clusters with operand multicast when the matrix has enough tiles to fill the device with them
    if (P.T >= 8) {
        constexpr int CLI = DIGITS == 1 ? DG_CMO_CLUSTER_I : DG_CLUSTER_I, CLJ = DG_CLUSTER_J;
        constexpr int TB = DIGITS == 1 ? 2 : 1;                                      // tiles per CTA and side
        const size_t smem = DGKernelCfg<DIGITS, TB>::SMEM;
        auto kern = drmsd_gram_kernel<DIGITS, CLI, CLJ, TB>;
        CLUSCO_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        cudaLaunchConfig_t cfg = {};
        cfg.blockDim = dim3(DG_THREADS);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = CLI * CLJ;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        cfg.gridDim = dim3((unsigned)(sms / (CLI * CLJ) * (CLI * CLJ)));
        int clusters = 0;
        CLUSCO_CUDA_TRY(cudaOccupancyMaxActiveClusters(&clusters, kern, &cfg));    // co-resident clusters
        P.n_sched = dg_schedule_count(P.T, TB * CLI, TB * CLJ);
        if (clusters > P.n_sched) clusters = (int)P.n_sched;
        if (clusters >= 1) {
            // blocks of about `clusters` super-tiles, square in tile units, so that a wave shares A rows and B columns in L2
            int32_t bj = 1;
            while ((int64_t)(bj + 1) * CLJ * (bj + 1) * CLJ <= (int64_t)clusters * CLI * CLJ) ++bj;
            const int32_t bi = (bj * CLJ + CLI - 1) / CLI;
            dg_schedule_kernel<<<1, 32, 0, s>>>(P.T, TB * CLI, TB * CLJ, bi, bj, (int2*)(ws + w.off_sched));
            CLUSCO_CUDA_TRY(cudaGetLastError());
            cfg.gridDim = dim3((unsigned)(clusters * CLI * CLJ));
            CLUSCO_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, P));
            return CLUSCO_OK;
        }
    }
    P.n_sched = 0;
    const size_t smem = DGKernelCfg<DIGITS, 1>::SMEM;
    CLUSCO_CUDA_TRY(cudaFuncSetAttribute(drmsd_gram_kernel<DIGITS, 1, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t grid = P.total < sms ? P.total : sms;
    drmsd_gram_kernel<DIGITS, 1, 1, 1><<<(unsigned)grid, DG_THREADS, smem, s>>>(P);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

}  // namespace clusco
