// common.cuh -- shared host/device helpers of libclusco (no arithmetic of the method lives here).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/clusco.h"

namespace clusco {

// ---- per-model record produced by the stats kernel and consumed by every Gram engine -------------
// The centred coordinates of model n are scaled by 2^-ex so that max |a| lies in [0.5, 1); S = sum of
// squares of the scaled fp32 values (accumulated in FP64, stored as a two-float sum Shi + Slo).
struct ModelStat {
    double mean[3];
    float Shi, Slo;
    int32_t ex;
    int32_t pad;
};

static inline int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

// thread-local last CUDA error for clusco_last_cuda_error()
extern thread_local int g_last_cuda_error;

#define CLUSCO_CUDA_TRY(expr)                                   \
    do {                                                        \
        cudaError_t _e = (expr);                                \
        if (_e != cudaSuccess) {                                \
            ::clusco::g_last_cuda_error = (int)_e;              \
            return CLUSCO_ERR_CUDA;                             \
        }                                                       \
    } while (0)

// packed row-major upper-triangle index of (i, j), i < j  (N(N-1)/2 values)
__host__ __device__ __forceinline__ int64_t packed_index(int64_t i, int64_t j, int64_t N)
{
    return i * (2 * N - i - 1) / 2 + (j - i - 1);
}

// exact 2^k as float for k in [-126, 127]
__device__ __forceinline__ float pow2i(int k) { return __int_as_float((k + 127) << 23); }

// per-model epilogue records of the tensor-core engine (gram_i8tc.cuh: I8_CSTAT_TILE floats per column tile of 16 models,
// [sum a^2 high | sum a^2 low | 2^e]); 16 bytes per model are reserved for them in the workspace
constexpr int64_t I8_RECORD_BYTES_PER_MODEL = 16;

// ---- what the fused all-pairs kernels do with a finished pair (i < j, c = cRMSD) ---------------------------
// STORE:    out[packed index]                                   (a5, the matrix itself)
// BELOW:    compacted (i, j, c) triples of the pairs with c < cutoff -- the paper's first use case filters the
//           full matrix for pairs below 3.2 A; the matrix is never written
// ROWSTATS: rowsum[i] += c, rowsum[j] += c and the neighbour counts below[.] += (c < cutoff) -- the per-model
//           reductions that representative selection consumes (mean cRMSD to the others)
enum SinkMode { SINK_STORE = 0, SINK_BELOW = 1, SINK_ROWSTATS = 2 };
struct Sink {
    float cutoff;
    int64_t capacity;               // BELOW: slots in pair_i / pair_j / pair_c
    int32_t* pair_i;
    int32_t* pair_j;
    float* pair_c;
    unsigned long long* count;      // BELOW: number of pairs found (may exceed capacity; extra pairs are dropped)
    double* rowsum;                 // ROWSTATS
    int32_t* below;
};

// one pair, no cooperation between threads (the CUDA-core engine and the ragged edges use this form)
template <int MODE>
__device__ __forceinline__ void sink_emit(const Sink& S, int32_t i, int32_t j, float c)
{
    if (MODE == SINK_BELOW) {
        if (c < S.cutoff) {
            const unsigned long long slot = atomicAdd(S.count, 1ull);
            if ((int64_t)slot < S.capacity) {
                S.pair_i[slot] = i;
                S.pair_j[slot] = j;
                S.pair_c[slot] = c;
            }
        }
    } else if (MODE == SINK_ROWSTATS) {
        atomicAdd(S.rowsum + i, (double)c);
        atomicAdd(S.rowsum + j, (double)c);
        if (c < S.cutoff) {
            atomicAdd(S.below + i, 1);
            atomicAdd(S.below + j, 1);
        }
    }
}

// ---- tensor-core engine geometry (gram_i8tc.cuh) ---------------------------------------------------
constexpr int I8_ROW_MODELS = 32;      // models per row tile: 4 TMEM quadrants x 8 models; lane = r + 8 p (p = 3: zero rows)
constexpr int I8_COL_MODELS = 16;      // models per column tile: MMA N = 3 x 16 = 48 per level block
constexpr int I8_A_SLAB = 128 * 32;    // bytes of one (k-step, digit) A slab: 128 rows x 32 atoms, int8
constexpr int I8_B_SLAB = 144 * 32;    // bytes of one k-step B slab: 3 digits x 48 rows x 32 atoms
constexpr int I8_MAX_KSTEPS = 8;       // L <= 256: a row tile's A operand (3 digits x ksteps x 8 columns) stays resident in TMEM

// ---- workspace layout --------------------------------------------------------------------------
// [ ModelStat[Np] | i8 epilogue records | FFMA plane | i8 A planes | i8 B planes ]      Np = N rounded up to 128
struct Workspace {
    int64_t N, Np;
    int32_t L;
    int32_t Lp16;        // L rounded up to 16 (FFMA k-chunk)
    int32_t Lp32;        // L rounded up to 32 (kind::i8 MMA K)
    int64_t row_tiles, col_tiles;   // i8 engine
    size_t off_stats, off_pstat, off_ffma, off_i8a, off_i8b, total;
};

static inline Workspace workspace_layout(int64_t N, int32_t L)
{
    Workspace w;
    w.N = N;
    w.L = L;
    w.Np = round_up(N, 128);
    w.Lp16 = (int32_t)round_up(L, 16);
    w.Lp32 = (int32_t)round_up(L, 32);
    w.row_tiles = (N + I8_ROW_MODELS - 1) / I8_ROW_MODELS;
    w.col_tiles = (N + I8_COL_MODELS - 1) / I8_COL_MODELS;
    size_t o = 0;
    w.off_stats = o;
    o += (size_t)round_up((int64_t)sizeof(ModelStat) * w.Np, 256);
    w.off_pstat = o;
    o += (size_t)round_up(I8_RECORD_BYTES_PER_MODEL * w.Np, 256);
    w.off_ffma = o;                                        // float Yt[Lp16][3*Np]
    o += (size_t)round_up((int64_t)sizeof(float) * w.Lp16 * 3 * w.Np, 256);
    const int64_t ks = w.Lp32 / 32;
    w.off_i8a = o;                                         // int8 Ap[row_tiles][ks][3][I8_A_SLAB]
    o += (size_t)round_up(w.row_tiles * ks * 3 * I8_A_SLAB, 256);
    w.off_i8b = o;                                         // int8 Bp[col_tiles][ks][I8_B_SLAB]
    o += (size_t)round_up(w.col_tiles * ks * I8_B_SLAB, 256);
    w.total = o;
    return w;
}

}  // namespace clusco
