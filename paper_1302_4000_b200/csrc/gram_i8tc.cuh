// gram_i8tc.cuh -- tensor-core engine of the all-pairs kernel: steps a3 (covariance), a4 (eq. 2 closed form) and
// a5 (packed store) fused in one persistent, warp-specialised kernel on tcgen05 (kind::i8) with int32
// accumulators in TMEM.
//
// Arithmetic: the centred coordinates of model n, scaled by 2^-ex_n so that max|a| is in
// [0.5, 1), are multiplied by KAPPA 2^23 (KAPPA = 127/128) and rounded to a 24-bit integer
//      I = d0 2^16 + d1 2^8 + d2,        d0, d1, d2 signed 8-bit digits (|d0| <= 127 thanks to KAPPA).
// The nine covariance sums of a pair are then  G = sum_k I_A I_B = 2^32 V0 + 2^24 V1 + 2^16 V2 (+ two
// dropped low-order levels),  V0 = d0.d0,  V1 = d0.d1 + d1.d0,  V2 = d0.d2 + d1.d1 + d2.d0: six int8 products,
// accumulated EXACTLY in int32.  The sums of squares of eq. 2's R^2 are taken from the same integers.
//
// Tile = 32 row models x 16 column models.  MMA view: A = [128 rows x K] with row (= TMEM lane) 32 w + 8 p + r
// holding component p of row model 8 w + r (p = 3: zero rows), B = [48 rows x K] per digit with row 16 q + o
// holding component q of column model (o & 1) * 4 + ((o >> 1) & 3) + (o & 8).  Per 32-atom k-step three MMAs
//      D[  0:144) += A(d0) . [B(d0); B(d1); B(d2)]^T      (levels 0, 1, 2)
//      D[ 48:144) += A(d1) . [B(d0); B(d1)]^T              (levels 1, 2)
//      D[ 96:144) += A(d2) . [B(d0)]^T                     (level 2)
// leave level v of (p, q, pair) at TMEM column 48 v + 16 q + o.  With this placement a 16x256b TMEM load hands
// every epilogue thread the three components p of ONE row model (lanes r, r+8, r+16) for two column models, so
// the nine sums of a pair meet in one thread without any shuffle.
//
// Roles (20 warps): one service warpgroup -- warp 0 = bulk-copy producer (operand planes are stored in HBM as
// shared-memory images in the canonical K-major core-matrix layout, so tiles arrive by plain 1-D cp.async.bulk),
// warp 1 = MMA issuer (one thread) and TMEM owner, warps 2, 3 idle -- that hands most of its registers to the four
// epilogue warpgroups (setmaxnreg); warps 4..19 = four epilogue teams of 4 warps (one per TMEM quadrant) that take the
// tiles in turn, each thread carrying four pairs of a tile (two packed groups, two independent dependency chains).
// TMEM accumulator buffers of 144 columns: three for L <= 160, two above; a row tile's A operand is moved once from a
// shared-memory staging area into TMEM (tcgen05.cp, columns after the buffers) and read from there by every MMA (for L in
// 97..160 some slabs of the third digit stay in the staging area, which is then double-buffered).  A team holds a
// buffer only while it loads and recombines the three levels; the closed form runs after the buffer has been handed
// back.  The epilogue's sink is a template parameter: packed store (a5), threshold compaction, or row statistics.
#pragma once
#include "common.cuh"
#include "epilogue.cuh"
#include "i8_layout.cuh"
#include "prep.cuh"
#include "tc_ptx.cuh"

namespace clusco {

__host__ __device__ constexpr int i8_a_stagings(int ks);
constexpr double I8_KAPPA = 127.0 / 128.0;
constexpr int I8_MAX_STAGES = 6;               // B stages (whole column tiles) in flight: as many as shared memory holds, up to this
constexpr int I8_ACC_COLS = 144;               // TMEM columns per accumulator buffer (3 levels x 48)
constexpr int I8_MAX_ACC_BUFS = 3;
// Accumulator buffers: three for L <= 160 (k-steps <= 5), two above.  With four epilogue teams of four warps a buffer is
// held twice as long as with two teams of eight, and two buffers then starve the tensor pipe (measured at L = 100:
// 3.38 ms with two buffers, 3.05 ms with three); three buffers fit beside the whole A tile for k-steps <= 3, and for
// k-steps 4 and 5 when 2 respectively 5 slabs of the A tile's third digit stay in shared memory (i8_a_tmem_slabs).
// k-steps 6..8 keep two buffers: 1-3 % slower than the two-team kernel it replaces at L = 161..224, equal at L = 250.
constexpr int I8_NB3_MAX_KS = 5;
__host__ __device__ constexpr int i8_acc_bufs(int ks) { return ks <= I8_NB3_MAX_KS ? 3 : 2; }
// (k-step, digit) slabs of the A tile kept in tensor memory, in the order digit-major; the remaining ones (the last
// k-steps of the third digit, if any) are read from the shared-memory staging area by their (narrow, N = 48) MMAs
__host__ __device__ constexpr int i8_a_tmem_slabs(int ks)
{
    return (512 - i8_acc_bufs(ks) * I8_ACC_COLS) / 8 < 3 * ks ? (512 - i8_acc_bufs(ks) * I8_ACC_COLS) / 8 : 3 * ks;
}
__host__ __device__ constexpr int i8_a_stagings(int ks) { return i8_a_tmem_slabs(ks) < 3 * ks ? 2 : 1; }
constexpr int I8_EPI_WARPS = 16;
constexpr int I8_EPI_TEAMS = 4;                // teams of four warps (one per TMEM quadrant) that take the tiles in turn
constexpr int I8_SERVICE_WARPS = 4;            // one warpgroup: bulk-copy producer, MMA issuer, two idle warps
// (the service warps take the LOWEST warp numbers: measured, waiting service warps with high numbers -- which issue first
// among a scheduler's ready warps -- cost the epilogue 4-12 % at L <= 96)
constexpr int I8_PRODUCER_WARP = 0, I8_MMA_WARP = 1;
constexpr int I8_THREADS = (I8_SERVICE_WARPS + I8_EPI_WARPS) * 32;
// Register split (setmaxnreg works on warpgroups of four warps and moves registers inside the CTA's own allocation): the
// kernel starts with 96 registers per thread (five warps per scheduler); the service warpgroup shrinks to
// I8_REGS_SERVICE, which frees 128 x (96 - 24) registers, and the four epilogue warpgroups grow to I8_REGS_EPI, which
// takes 512 x (112 - 96) <= that.  (Asking for more than was freed never completes: the increase waits for registers.)
constexpr int I8_REGS_SERVICE = 24;
constexpr int I8_REGS_EPI = 112;
static_assert(I8_EPI_WARPS * (I8_REGS_EPI - 96) <= I8_SERVICE_WARPS * (96 - I8_REGS_SERVICE), "register split must balance");
constexpr int I8_HIT_CAP = 64;                 // BELOW: hits staged per epilogue warp before one atomic reserves their slots
constexpr size_t I8_HIT_BYTES = (size_t)I8_EPI_WARPS * I8_HIT_CAP * 12;

static inline bool i8tc_supported(int32_t L) { return L >= 1 && L <= 32 * I8_MAX_KSTEPS; }

// ---- a1 + a2 + operand planes, one launch --------------------------------------------------------------------
// Ap[row_tile][digit][kstep][I8_A_SLAB], Bp[col_tile][kstep][I8_B_SLAB]; a slab is a grid of 8-row x 16-byte core
// matrices: byte (row, k) of a slab sits at (row/8)*256 + (k/16)*128 + (row%8)*16 + k%16  (i8_layout.cuh, whose functions
// a host harness shares with this kernel: tests/test_i8_layout.py).
// One warp per model slot.  The model is read ONCE, element-wise (coalesced), and stays in registers through
// three passes: FP64 centroid -> max|a| (scale exponent) -> fixed-point integers I.  The integers of a round
// (4 k-steps = 128 atoms) go through a warp-private shared-memory strip so that each lane can pack the digit
// bytes of 4 consecutive atoms of one component into one 32-bit store of the operand images.
// Per-model records the epilogue reads (sum of squares as two floats, scale 2^e), stored per column tile of 16 models as
// [Thi[16] | Tlo[16] | pw[16]] with model m of the tile at slot i8_col_slot(m) -- the order of the B rows -- so that the
// two column models of an epilogue thread (c and c + 4) are adjacent: one 8-byte load per quantity.
constexpr int I8_CSTAT_TILE = 48;
constexpr int I8_PREP_WARPS = 8;
constexpr int I8_PREP_STRIP = 4 * 97;          // ints per warp and round: 4 k-steps x (96 + 1 pad)

__global__ void __launch_bounds__(I8_PREP_WARPS * 32) i8_prep_kernel(const float* __restrict__ coords, int64_t N, int32_t L,
                                                                     int32_t ks, int64_t row_slots, int64_t col_slots,
                                                                     int64_t stat_slots, int8_t* __restrict__ Ap,
                                                                     int8_t* __restrict__ Bp, float* __restrict__ cstat)
{
    __shared__ int strip_s[I8_PREP_WARPS][I8_PREP_STRIP];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t n = (int64_t)blockIdx.x * I8_PREP_WARPS + wib;
    if (n >= stat_slots) return;
    const bool valid = n < N;
    const int n_el = valid ? 3 * L : 0;
    const float* x = coords + n * (int64_t)L * 3;
    // element e = 384 r + 32 t + lane of the model; its component is (2 t + lane) % 3  (384 and 30 t are multiples of 3)
    const int l3 = lane % 3;
    float v[2][12];
    double acc[3] = {0.0, 0.0, 0.0};                       // acc[q]: component (q + l3) % 3, q = (2 t) % 3
    bool finite = true;
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int t = 0; t < 12; ++t) {
            const int e = 384 * r + 32 * t + lane;
            const float xv = e < n_el ? x[e] : 0.0f;
            v[r][t] = xv;
            finite = finite && (fabsf(xv) <= 3.0e38f);
            acc[(2 * t) % 3] += (double)xv;
        }
    // per-component sums: lane holds component c in acc[(c - l3 + 3) % 3]
    double mean[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int q = (c - l3 + 3) % 3;
        const double mine = q == 0 ? acc[0] : (q == 1 ? acc[1] : acc[2]);
        mean[c] = warp_sum(mine) / (double)L;
    }
    double mq[3];                                          // centroid component matching acc[q]
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const int c = (q + l3) % 3;
        mq[q] = c == 0 ? mean[0] : (c == 1 ? mean[1] : mean[2]);
    }
    float amax = 0.0f;
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int t = 0; t < 12; ++t)
            if (384 * r + 32 * t + lane < n_el) amax = fmaxf(amax, fabsf((float)((double)v[r][t] - mq[(2 * t) % 3])));
    amax = warp_max(amax);
    int ex = 0;
    if (amax > 0.0f && amax < 3.0e38f) (void)frexpf(amax, &ex);          // amax = m 2^ex, m in [0.5, 1)
    const bool finite_range = ex <= 30;                    // coordinates beyond 2^30 Angstrom are not representable
    ex = max(-30, min(30, ex));
    const double scale = valid ? ldexp(I8_KAPPA, 23 - ex) : 0.0;

    // (A image: row tile n/32, quadrant w = (n%32)/8, row-in-group r = n%8, row group 4w + p; B image: column tile n/16,
    // o = position of this model among the 16 columns of a component block -- i8_store_lane_words)
    const int64_t b_tile = n >> 4;
    const int m16 = (int)(n & 15);
    const int sub = lane >> 3, j = lane & 7;               // packing role: k-step 4 r + sub, atoms 4 j .. 4 j + 3 of it
    int* strip = strip_s[wib];
    unsigned long long sumsq = 0ull;
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        if (4 * r >= ks) break;                            // warp-uniform
#pragma unroll
        for (int t = 0; t < 12; ++t) {
            const int el = 32 * t + lane;                  // element within the round
            int I = 0;
            if (384 * r + el < n_el) I = __double2int_rn(((double)v[r][t] - mq[(2 * t) % 3]) * scale);
            sumsq += (unsigned long long)((long long)I * (long long)I);
            strip[el + el / 96] = I;
        }
        __syncwarp();
        const int kk = 4 * r + sub;
        if (kk < ks) {
#pragma unroll
            for (int p = 0; p < 3; ++p) {
                uint32_t w[3] = {0u, 0u, 0u};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    int d0, d1, d2;
                    i8_digits(strip[97 * sub + 3 * (4 * j + i) + p], d0, d1, d2);
                    w[0] |= (uint32_t)(d0 & 0xff) << (8 * i);
                    w[1] |= (uint32_t)(d1 & 0xff) << (8 * i);
                    w[2] |= (uint32_t)(d2 & 0xff) << (8 * i);
                }
                i8_store_lane_words(Ap, Bp, n < row_slots, n < col_slots, n, ks, kk, j, p, w[0], w[1], w[2]);
            }
            i8_store_lane_words(Ap, Bp, n < row_slots, false, n, ks, kk, j, 3, 0u, 0u, 0u);      // the zero rows
        }
        __syncwarp();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sumsq += __shfl_xor_sync(0xffffffffu, sumsq, o);
    finite = __all_sync(0xffffffffu, finite);
    if (lane == 0) {
        const double T = ldexp((double)sumsq, 2 * ex - 46);          // KAPPA^2 sum |a|^2, Angstrom^2
        float Thi = (float)T;
        const float Tlo = (float)(T - (double)Thi);
        if (!finite || !finite_range) Thi = __int_as_float(0x7fc00000);     // NaN/Inf coordinates poison this model's pairs
        float* rec = cstat + b_tile * I8_CSTAT_TILE + i8_stat_slot(m16);
        rec[0] = Thi;
        rec[16] = Tlo;
        rec[32] = pow2i(ex);
    }
}

// ---- tile walk ----------------------------------------------------------------------------------------------
// Row tile I (32 models) meets column tiles J = 2I .. Tc-1 (16 models each).  Tiles of the call's row-tile range
// [I_lo, I_hi) are linearised row-major; CTA b owns the contiguous range [total b / G, total (b+1) / G).
struct I8Tiles {
    int64_t Tc, I_lo, I_hi, total;
};
__host__ __device__ __forceinline__ int64_t i8_tiles_before(const I8Tiles& t, int64_t I)
{
    return (I - t.I_lo) * t.Tc - (I * (I - 1) - t.I_lo * (t.I_lo - 1));
}
__device__ __forceinline__ void i8_tile_from_linear(const I8Tiles& t, int64_t lin, int64_t& I, int64_t& J)
{
    int64_t lo = t.I_lo, hi = t.I_hi - 1;                  // largest I with tiles_before(I) <= lin
    while (lo < hi) {
        const int64_t mid = (lo + hi + 1) >> 1;
        if (i8_tiles_before(t, mid) <= lin) lo = mid; else hi = mid - 1;
    }
    I = lo;
    J = 2 * I + (lin - i8_tiles_before(t, I));
}

struct I8Params {
    const int8_t* Ap;
    const int8_t* Bp;
    const float* cstat;    // per-model records, I8_CSTAT_TILE floats per column tile (see i8_prep_kernel)
    float* out;
    int64_t N, row_begin, row_end, base;
    int32_t stages;        // B ring depth (one stage = the whole column tile, KS k-steps)
    float invLk;           // 1 / (KAPPA^2 L)
    I8Tiles tiles;
    Sink sink;             // MODE != SINK_STORE: where finished pairs go instead of `out`
};

// KS = k-steps (32 atoms each) per model, a template parameter so that the 3 KS MMAs of a tile are issued as
// straight-line code with immediate operand offsets: the issuing warp is the critical resource of this kernel
// (3 MMAs of 72 + 48 + 24 tensor cycles per k-step leave ~48 cycles of issue time per MMA).
// MODE (SinkMode) selects what the epilogue does with a finished pair: packed store (a5), threshold compaction or
// per-model row statistics (the fused consumers of the matrix).
template <int KS, int MODE>
__global__ void __launch_bounds__(I8_THREADS, 1) gram_i8tc_kernel(const I8Params P)
{
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr uint32_t STAGE_BYTES = KS * I8_B_SLAB;
    const int stages = P.stages;
    constexpr int NB = i8_acc_bufs(KS);
    constexpr int AS = i8_a_tmem_slabs(KS);                      // slabs of the A tile resident in tensor memory
    static_assert(NB * I8_ACC_COLS + 8 * AS <= 512 && AS >= 2 * KS, "tensor memory budget");
    // A staging: one area when the whole tile moves on into tensor memory, two (used alternately) when some slabs are read
    // from it for the whole row tile -- so that the next row tile's A still arrives while the current one is in use
    constexpr int NA = i8_a_stagings(KS);
    constexpr uint32_t A_BYTES = 3u * KS * I8_A_SLAB;
    uint8_t* sA = smem;                                          // NA x 3 digits x KS x 4096
    uint8_t* sB = smem + (size_t)NA * A_BYTES;                   // stages x KS x 4608
    uint64_t* bars = reinterpret_cast<uint64_t*>(sB + (size_t)stages * STAGE_BYTES);
    // barrier map: [0,S) b_full, [S,2S) b_empty, 2S.. a_full[2], a_empty[2], 2S+4.. acc_full[4] (one per epilogue TEAM: a
    // waiter must see every phase of its barrier, and a team meets a given buffer only every second or third use),
    // 2S+8.. acc_empty[3] (one per buffer; the MMA warp sees every phase)
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto B_FULL = [&](uint32_t s) { return bar0 + 8u * s; };
    auto B_EMPTY = [&](uint32_t s) { return bar0 + 8u * (stages + s); };
    auto A_FULL = [&](uint32_t a) { return bar0 + 8u * (2 * stages + a); };
    auto A_EMPTY = [&](uint32_t a) { return bar0 + 8u * (2 * stages + 2 + a); };
    auto ACC_FULL = [&](uint32_t t) { return bar0 + 8u * (2 * stages + 4 + t); };
    auto ACC_EMPTY = [&](uint32_t b) { return bar0 + 8u * (2 * stages + 4 + I8_EPI_TEAMS + b); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * stages + 4 + I8_EPI_TEAMS + I8_MAX_ACC_BUFS);

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            ptx::mbar_init(B_FULL(s), 1);
            ptx::mbar_init(B_EMPTY(s), 1);
        }
        for (int a = 0; a < NA; ++a) {
            ptx::mbar_init(A_FULL(a), 1);
            ptx::mbar_init(A_EMPTY(a), 1);
        }
        for (int t = 0; t < I8_EPI_TEAMS; ++t) ptx::mbar_init(ACC_FULL(t), 1);
        for (int b = 0; b < NB; ++b) ptx::mbar_init(ACC_EMPTY(b), I8_EPI_WARPS / I8_EPI_TEAMS);
        ptx::fence_mbar_init();
    }
    if (warp == I8_MMA_WARP) ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    const int64_t G = gridDim.x, b = blockIdx.x;
    const int64_t t0 = P.tiles.total * b / G, t1 = P.tiles.total * (b + 1) / G;
    const int64_t Tc = P.tiles.Tc;
    const uint32_t ntiles = (uint32_t)(t1 - t0);
    int64_t I0, J0;
    i8_tile_from_linear(P.tiles, t0, I0, J0);

    if (warp < I8_SERVICE_WARPS) {
    ptx::setmaxnreg_dec<I8_REGS_SERVICE>();
    if (warp == I8_PRODUCER_WARP) {
        // ===== producer: one elected lane streams operand images with 1-D bulk copies =====
        if (lane == 0) {
            int64_t I = I0, J = J0;
            int64_t curI = -1;
            uint32_t a_loads = 0, stage = 0, phase = 0;
            for (uint32_t n = 0; n < ntiles; ++n) {
                if (I != curI) {
                    const uint32_t a = a_loads % NA;             // load number a_loads / NA of that staging area
                    ptx::mbar_wait(A_EMPTY(a), ((a_loads / NA) & 1) ^ 1);
                    ptx::mbar_expect_tx(A_FULL(a), A_BYTES);
                    ptx::bulk_g2s(ptx::smem_u32(sA + (size_t)a * A_BYTES), P.Ap + (size_t)I * A_BYTES, A_BYTES, A_FULL(a));
                    ++a_loads;
                    curI = I;
                }
                ptx::mbar_wait(B_EMPTY(stage), phase ^ 1);
                ptx::mbar_expect_tx(B_FULL(stage), STAGE_BYTES);
                ptx::bulk_g2s(ptx::smem_u32(sB + (size_t)stage * STAGE_BYTES), P.Bp + (size_t)J * STAGE_BYTES, STAGE_BYTES,
                              B_FULL(stage));
                if (++stage == (uint32_t)stages) { stage = 0; phase ^= 1; }
                if (++J >= Tc) { ++I; J = 2 * I; }
            }
        }
    } else if (warp == I8_MMA_WARP) {
        // ===== MMA issuer: the whole warp walks the loop (warp-uniform control flow and addresses, so the
        // operands live in uniform registers); one elected lane issues =====
        constexpr uint32_t ID144 = ptx::idesc_s8(128, 144), ID96 = ptx::idesc_s8(128, 96), ID48 = ptx::idesc_s8(128, 48);
        // descriptor = hi word (SBO 256 B, version 1) | lo word (LBO 128 B, start address >> 4)
        constexpr uint64_t DESC_HI = (uint64_t)((256u >> 4) | (1u << 14)) << 32;
        uint32_t a_lo0 = 0;                                      // descriptor low word of the current row tile's staging area
        const uint32_t b_lo0 = ((128u >> 4) << 16) | ((ptx::smem_u32(sB) & 0x3FFFFu) >> 4);
        const uint32_t a_tm = tmem + NB * I8_ACC_COLS;           // digit a, k-step k at column 8 (a KS + k)
        uint32_t rem = 0;                                        // tiles left in the current row tile
        uint32_t next_rem = (uint32_t)(Tc - J0);
        uint32_t next_row_len = (uint32_t)(Tc - 2 * (I0 + 1));   // each further row is two tiles shorter
        uint32_t a_uses = 0, stage = 0, phase = 0;
        uint32_t buf = 0, acc_par = 0;                           // tile n: buffer n % NB, use number n / NB of it
        for (uint32_t n = 0; n < ntiles; ++n) {
            if (rem == 0) {
                // new row tile: move its A operand from the shared-memory staging area into tensor memory
                // (tcgen05.cp runs in order with the MMAs, so the previous row's MMAs are done reading)
                rem = next_rem;
                next_rem = next_row_len;
                next_row_len -= 2;
                const uint32_t a = a_uses % NA;
                ptx::mbar_wait(A_FULL(a), (a_uses / NA) & 1);
                ptx::tc_fence_after();
                a_lo0 = ((128u >> 4) << 16) | ((ptx::smem_u32(sA + (size_t)a * A_BYTES) & 0x3FFFFu) >> 4);
                if (ptx::elect_one()) {
#pragma unroll
                    for (int s = 0; s < AS; ++s)
                        ptx::tmem_cp_128x256b(a_tm + 8 * s, DESC_HI | (a_lo0 + s * (I8_A_SLAB >> 4)));
                    if (AS == 3 * KS) ptx::tc_commit(A_EMPTY(a));  // staging area free once the copies are done
                }
                __syncwarp();
                ++a_uses;
            }
            --rem;
            ptx::mbar_wait(ACC_EMPTY(buf), acc_par ^ 1);
            ptx::mbar_wait(B_FULL(stage), phase);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
                const uint32_t d = tmem + buf * I8_ACC_COLS;
                const uint32_t b_lo = b_lo0 + stage * (STAGE_BYTES >> 4);
#pragma unroll
                for (int k = 0; k < KS; ++k) {
                    const uint64_t db = DESC_HI | (b_lo + k * (I8_B_SLAB >> 4));
                    ptx::mma_i8_ts(d, a_tm + 8 * k, db, ID144, k > 0);
                    ptx::mma_i8_ts(d + 48, a_tm + 8 * (KS + k), db, ID96, 1);
                    if (2 * KS + k < AS)
                        ptx::mma_i8_ts(d + 96, a_tm + 8 * (2 * KS + k), db, ID48, 1);
                    else
                        ptx::mma_i8(d + 96, DESC_HI | (a_lo0 + (2 * KS + k) * (I8_A_SLAB >> 4)), db, ID48, 1);
                }
                ptx::tc_commit(B_EMPTY(stage));
                ptx::tc_commit(ACC_FULL(n % I8_EPI_TEAMS));
                // third digit read from the staging area: it is free only after the row tile's last MMA
                if (AS < 3 * KS && rem == 0) ptx::tc_commit(A_EMPTY((a_uses - 1) % NA));
            }
            __syncwarp();
            if (++stage == (uint32_t)stages) { stage = 0; phase ^= 1; }
            if (++buf == (uint32_t)NB) { buf = 0; acc_par ^= 1; }
        }
    }
    } else {
        ptx::setmaxnreg_inc<I8_REGS_EPI>();
        // ===== epilogue =====
        // Four teams of four warps (one per TMEM quadrant) take the tiles in turn.  A thread owns FOUR pairs of a tile: row
        // model r of its quadrant against column models c, c + 4 (column half 0) and c + 8, c + 12 (half 1) -- two packed
        // (float2) groups that go through the closed form as two independent dependency chains, and that share the
        // per-tile bookkeeping (barrier, tile walk, addresses) and the TMEM loads (16x256b.x2 spans both halves).
        const int ew = warp - I8_SERVICE_WARPS;
        const int team = ew >> 2;                                // 0 .. I8_EPI_TEAMS - 1
        const int quad = warp & 3;                               // TMEM lanes 32 quad .. 32 quad + 31
        const int r = lane >> 2, c4 = lane & 3;
        // tile coordinates and model indices fit 32 bits (N <= 2^24); only the packed offset needs 64
        const int32_t Tc32 = (int32_t)Tc, N32 = (int32_t)P.N;
        int32_t I = (int32_t)I0, J = (int32_t)J0;
        for (int s = 0; s < team; ++s)
            if (++J >= Tc32) { ++I; J = 2 * I; }
        int32_t curI = -1, i = 0;
        int64_t rowoff = 0;
        bool row_ok = false;
        float si_Thi = 0.0f, si_Tlo = 0.0f, si_pw = 1.0f;          // row model's record
        // ROWSTATS: running sum / count of the row this lane group is on (rows persist over consecutive tiles)
        double acc_sum = 0.0;
        int32_t acc_cnt = 0, acc_i = -1;
        // BELOW: hits are staged per warp in shared memory and appended I8_HIT_CAP at a time -- ONE atomic on the shared
        // counter per flush (a single hot address serialises in L2: one atomic per warp and tile cost +30 % at C3)
        uint8_t* hit_base = reinterpret_cast<uint8_t*>(tmem_slot) + 16 + (size_t)ew * I8_HIT_CAP * 12;
        int32_t* hit_i = reinterpret_cast<int32_t*>(hit_base);
        int32_t* hit_j = hit_i + I8_HIT_CAP;
        float* hit_c = reinterpret_cast<float*>(hit_j + I8_HIT_CAP);
        int nhit = 0;                                            // warp-uniform
        auto flush_hits = [&]() {
            if (nhit == 0) return;
            __syncwarp();
            unsigned long long base = 0ull;
            if (lane == 0) base = atomicAdd(P.sink.count, (unsigned long long)nhit);
            base = __shfl_sync(0xffffffffu, base, 0);
            for (int e = lane; e < nhit; e += 32) {
                const int64_t slot = (int64_t)base + e;
                if (slot < P.sink.capacity) {
                    P.sink.pair_i[slot] = hit_i[e];
                    P.sink.pair_j[slot] = hit_j[e];
                    P.sink.pair_c[slot] = hit_c[e];
                }
            }
            __syncwarp();
            nhit = 0;
        };
        auto flush_row = [&]() {
            if (c4 == 0 && acc_i >= 0 && acc_i < (int32_t)P.N) {
                atomicAdd(P.sink.rowsum + acc_i, acc_sum);
                if (acc_cnt) atomicAdd(P.sink.below + acc_i, acc_cnt);
            }
        };
        uint32_t buf = (uint32_t)team % NB, full_par = 0;       // this team's tile n: buffer n % NB; visit n / 4 of the team
        for (uint32_t n = team; n < ntiles; n += I8_EPI_TEAMS) {
            if (I != curI) {                                     // per-row quantities (warp-uniform branch)
                curI = I;
                i = I * I8_ROW_MODELS + quad * 8 + r;
                row_ok = i < N32 && i >= (int32_t)P.row_begin && i < (int32_t)P.row_end;
                const float* ri = P.cstat + (size_t)(i >> 4) * I8_CSTAT_TILE + i8_stat_slot(i & 15);   // slots beyond N hold neutral records
                // (the identity shuffles make the warp wait for these three loads HERE, in the rare row-change path: left
                // pending, their scoreboard slot is shared with the per-tile loads below and the first read of si_* in
                // every later tile then waits for those)
                si_Thi = __shfl_sync(0xffffffffu, ri[0], lane);
                si_Tlo = __shfl_sync(0xffffffffu, ri[16], lane);
                si_pw = __shfl_sync(0xffffffffu, ri[32], lane);
                rowoff = (int64_t)i * (2 * P.N - i - 1) / 2 - i - 1 - P.base;
            }
            const int32_t j0 = J * I8_COL_MODELS + c4;           // this thread's column models: j0, j0 + 4, j0 + 8, j0 + 12
            // their records: one 16-byte load per quantity, in the order (j0, j0 + 4 | j0 + 8, j0 + 12) of the two groups;
            // first used in the last line of eq. 2, a whole closed form away
            const float* cj = P.cstat + (size_t)J * I8_CSTAT_TILE + c4 * 4;
            const float4 Thj = *reinterpret_cast<const float4*>(cj);
            const float4 Tlj = *reinterpret_cast<const float4*>(cj + 16);
            const float4 pwj = *reinterpret_cast<const float4*>(cj + 32);
            float* const dst = P.out + rowoff + j0;
            bool ok[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) ok[e] = row_ok && j0 + 4 * e < N32 && j0 + 4 * e > i;   // masked pairs are not stored
            const int32_t i_cur = i;
            // advance to the team's next tile (four tiles on)
#pragma unroll
            for (int s = 0; s < 4; ++s)
                if (++J >= Tc32) { ++I; J = 2 * I; }

            ptx::mbar_wait(ACC_FULL(team), full_par);
            full_par ^= 1;
            ptx::tc_fence_after();
            const uint32_t ta = tmem + ((uint32_t)(quad * 32) << 16) + buf * I8_ACC_COLS;
            // m[g][3p+q] = (.x, .y): pairs (row model r, column models c4 + 8 g and c4 + 8 g + 4); Gram sums in units of
            // 2^46.  The accumulator buffer is held only for the loads and the level recombination and handed back to the
            // MMA warp before any of the closed form runs (at L <= 128 the epilogue, not the tensor pipe, sets the pace).
            float2 m[2][9];
            {
                const float2 s30 = make_float2(0x1p-30f, 0x1p-30f), s14 = make_float2(0x1p-14f, 0x1p-14f);
                // register slots of a 16x256b.x2 load: [0,1] = lane r, half 0; [2,3] = lane r + 8, half 0; [4..7] the same
                // for half 1; lane window h = 0: p = 0 (lane r), p = 1 (lane r + 8); h = 1: p = 2 (lane r + 16), zero rows
                uint32_t v1[2][8], v2[2][8], v0[2][8];
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    // levels 1 and 2 first: T = 2^8 V1 + V2 fits int32 (|T| < 2^31 for L <= 256 because |d0| <= 127)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        ptx::tmem_ld_16x256b_x2(ta + ((uint32_t)(16 * h) << 16) + 48 + 16 * q, v1[h]);
                        ptx::tmem_ld_16x256b_x2(ta + ((uint32_t)(16 * h) << 16) + 96 + 16 * q, v2[h]);
                    }
                    ptx::tmem_ld_wait();
                    // level 0 is requested before levels 1 and 2 are converted, so its latency is covered by that work
#pragma unroll
                    for (int h = 0; h < 2; ++h) ptx::tmem_ld_16x256b_x2(ta + ((uint32_t)(16 * h) << 16) + 16 * q, v0[h]);
                    auto T = [&](int h, int e) { return (float)(((int32_t)v1[h][e] << 8) + (int32_t)v2[h][e]); };
#pragma unroll
                    for (int g = 0; g < 2; ++g) {
                        m[g][0 + q] = __fmul2_rn(make_float2(T(0, 4 * g + 0), T(0, 4 * g + 1)), s30);
                        m[g][3 + q] = __fmul2_rn(make_float2(T(0, 4 * g + 2), T(0, 4 * g + 3)), s30);
                        m[g][6 + q] = __fmul2_rn(make_float2(T(1, 4 * g + 0), T(1, 4 * g + 1)), s30);
                    }
                    ptx::tmem_ld_wait();
                    auto F = [&](int h, int e) { return (float)(int32_t)v0[h][e]; };
#pragma unroll
                    for (int g = 0; g < 2; ++g) {
                        m[g][0 + q] = __ffma2_rn(make_float2(F(0, 4 * g + 0), F(0, 4 * g + 1)), s14, m[g][0 + q]);
                        m[g][3 + q] = __ffma2_rn(make_float2(F(0, 4 * g + 2), F(0, 4 * g + 3)), s14, m[g][3 + q]);
                        m[g][6 + q] = __ffma2_rn(make_float2(F(1, 4 * g + 0), F(1, 4 * g + 1)), s14, m[g][6 + q]);
                    }
                }
                // the accumulator buffer is free again
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(ACC_EMPTY(buf));
                buf += I8_EPI_TEAMS % NB;                        // the team's next tile is four tiles on
                if (buf >= (uint32_t)NB) buf -= NB;
            }
            // the closed form, two independent chains (one per group of two pairs)
            float c[4];
            {
                const float2 Ti = make_float2(si_Thi, si_Thi), Tli = make_float2(si_Tlo, si_Tlo), pwi = make_float2(si_pw, si_pw);
                const EqInvariants<float2> inv0 = eq2_invariants(m[0]), inv1 = eq2_invariants(m[1]);
                const float2 c01 = eq2_finish(eq2_energy(inv0), Ti, Tli, pwi, make_float2(Thj.x, Thj.y),
                                              make_float2(Tlj.x, Tlj.y), make_float2(pwj.x, pwj.y), P.invLk);
                const float2 c23 = eq2_finish(eq2_energy(inv1), Ti, Tli, pwi, make_float2(Thj.z, Thj.w),
                                              make_float2(Tlj.z, Tlj.w), make_float2(pwj.z, pwj.w), P.invLk);
                c[0] = c01.x; c[1] = c01.y; c[2] = c23.x; c[3] = c23.y;
            }
            if (MODE == SINK_STORE) {
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    if (ok[e]) dst[4 * e] = c[e];
            } else if (MODE == SINK_BELOW) {
                // two batches of at most 64 candidates (one per group), so that I8_HIT_CAP = 64 slots always suffice
#pragma unroll
                for (int g = 0; g < 2; ++g) {
                    const bool h0 = ok[2 * g] && c[2 * g] < P.sink.cutoff, h1 = ok[2 * g + 1] && c[2 * g + 1] < P.sink.cutoff;
                    const uint32_t m0 = __ballot_sync(0xffffffffu, h0), m1 = __ballot_sync(0xffffffffu, h1);
                    const int add = __popc(m0) + __popc(m1);
                    if (add) {
                        if (nhit + add > I8_HIT_CAP) flush_hits();
                        const uint32_t lt = (1u << lane) - 1u;
                        if (h0) {
                            const int k = nhit + __popc(m0 & lt);
                            hit_i[k] = i_cur; hit_j[k] = j0 + 8 * g; hit_c[k] = c[2 * g];
                        }
                        if (h1) {
                            const int k = nhit + __popc(m0) + __popc(m1 & lt);
                            hit_i[k] = i_cur; hit_j[k] = j0 + 8 * g + 4; hit_c[k] = c[2 * g + 1];
                        }
                        nhit += add;
                    }
                }
            } else {
                // the warp holds 8 rows (r) x 16 columns (c4 + 4 e): reduce over the columns for the row sums (kept in
                // registers until the row changes) and over the rows for the column sums
                float cv[4];
                int32_t bc[2] = {0, 0};                          // below-counts of columns (0, 1) and (2, 3), 16 bits each
                float rs = 0.0f;
                int32_t rb = 0;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    cv[e] = ok[e] ? c[e] : 0.0f;
                    const int32_t b = ok[e] && c[e] < P.sink.cutoff ? 1 : 0;
                    rs += cv[e];
                    rb += b;
                    bc[e >> 1] |= b << (16 * (e & 1));
                }
#pragma unroll
                for (int o = 1; o <= 2; o <<= 1) {
                    rs += __shfl_xor_sync(0xffffffffu, rs, o);
                    rb += __shfl_xor_sync(0xffffffffu, rb, o);
                }
                if (i_cur != acc_i) {
                    flush_row();
                    acc_i = i_cur;
                    acc_sum = 0.0;
                    acc_cnt = 0;
                }
                acc_sum += (double)rs;
                acc_cnt += rb;
#pragma unroll
                for (int o = 4; o <= 16; o <<= 1) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) cv[e] += __shfl_xor_sync(0xffffffffu, cv[e], o);
                    bc[0] += __shfl_xor_sync(0xffffffffu, bc[0], o);
                    bc[1] += __shfl_xor_sync(0xffffffffu, bc[1], o);
                }
                if (r == 0) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int32_t j = j0 + 4 * e;
                        const int32_t b = (bc[e >> 1] >> (16 * (e & 1))) & 0xffff;
                        if (j < (int32_t)P.N) {
                            atomicAdd(P.sink.rowsum + j, (double)cv[e]);
                            if (b) atomicAdd(P.sink.below + j, b);
                        }
                    }
                }
            }
        }
        if (MODE == SINK_ROWSTATS) flush_row();
        if (MODE == SINK_BELOW) flush_hits();
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == I8_MMA_WARP) ptx::tmem_dealloc(tmem, 512);
}

static inline size_t i8tc_smem_bytes(int ks, int stages)
{
    return (size_t)i8_a_stagings(ks) * 3 * ks * I8_A_SLAB + (size_t)stages * ks * I8_B_SLAB +
           8 * (2 * stages + 4 + I8_EPI_TEAMS + I8_MAX_ACC_BUFS) + 16;
}
static inline int i8tc_stages(int ks, size_t extra)
{
    int st = I8_MAX_STAGES;
    while (st > 2 && i8tc_smem_bytes(ks, st) + extra > 227 * 1024) --st;
    return st;
}

static inline int i8tc_prepare(const float* coords, int64_t N, int32_t L, const Workspace& w, char* ws, cudaStream_t s)
{
    if (!i8tc_supported(L)) return CLUSCO_ERR_INVALID_ARG;
    const int ks = w.Lp32 / 32;
    const int64_t row_slots = w.row_tiles * I8_ROW_MODELS, col_slots = w.col_tiles * I8_COL_MODELS;
    i8_prep_kernel<<<(unsigned)((w.Np + I8_PREP_WARPS - 1) / I8_PREP_WARPS), I8_PREP_WARPS * 32, 0, s>>>(
        coords, N, L, ks, row_slots, col_slots, w.Np, (int8_t*)(ws + w.off_i8a), (int8_t*)(ws + w.off_i8b),
        (float*)(ws + w.off_pstat));
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

template <int MODE>
static inline int i8tc_compute(int64_t N, int32_t L, int64_t row_begin, int64_t row_end, float* out, const Sink& sink,
                               const Workspace& w, char* ws, int sms, cudaStream_t s)
{
    if (!i8tc_supported(L)) return CLUSCO_ERR_INVALID_ARG;
    I8Params P;
    P.Ap = (const int8_t*)(ws + w.off_i8a);
    P.Bp = (const int8_t*)(ws + w.off_i8b);
    P.cstat = (const float*)(ws + w.off_pstat);
    P.out = out;
    P.sink = sink;
    P.N = N;
    P.row_begin = row_begin;
    P.row_end = row_end;
    P.base = packed_index(row_begin, row_begin + 1, N);
    const int ks = w.Lp32 / 32;
    P.invLk = (float)(1.0 / (I8_KAPPA * I8_KAPPA * (double)L));
    P.tiles.Tc = w.col_tiles;
    P.tiles.I_lo = row_begin / I8_ROW_MODELS;
    P.tiles.I_hi = (row_end + I8_ROW_MODELS - 1) / I8_ROW_MODELS;
    P.tiles.total = i8_tiles_before(P.tiles, P.tiles.I_hi);
    if (P.tiles.total <= 0) return CLUSCO_OK;
    const size_t extra = MODE == SINK_BELOW ? I8_HIT_BYTES + 16 : 0;       // per-warp hit staging after the barriers
    P.stages = i8tc_stages(ks, extra);
    const size_t smem = i8tc_smem_bytes(ks, P.stages) + extra;
    const int64_t grid = P.tiles.total < sms ? P.tiles.total : sms;
    switch (ks) {
#define I8_LAUNCH(KS)                                                                                                  \
    case KS:                                                                                                           \
        CLUSCO_CUDA_TRY(cudaFuncSetAttribute(gram_i8tc_kernel<KS, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,  \
                                             (int)smem));                                                              \
        gram_i8tc_kernel<KS, MODE><<<(unsigned)grid, I8_THREADS, smem, s>>>(P);                                        \
        break;
        I8_LAUNCH(1) I8_LAUNCH(2) I8_LAUNCH(3) I8_LAUNCH(4) I8_LAUNCH(5) I8_LAUNCH(6) I8_LAUNCH(7) I8_LAUNCH(8)
#undef I8_LAUNCH
        default: return CLUSCO_ERR_INVALID_ARG;
    }
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

}  // namespace clusco
