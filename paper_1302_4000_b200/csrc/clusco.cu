// clusco.cu -- the C ABI declared in include/clusco.h: argument validation, workspace carving and kernel
// launches.  Every step of the path runs in the kernels of this directory; there is no CPU fallback.
#include <math.h>
#include <string.h>

#include <mutex>

#include "common.cuh"
#include "epilogue.cuh"
#include "gdt_ova.cuh"
#include "gram_ffma.cuh"
#include "drmsd_i8tc.cuh"
#include "gram_i8tc.cuh"
#include "one_vs_all.cuh"
#include "prep.cuh"
#include "ref_ova.cuh"

namespace clusco {
thread_local int g_last_cuda_error = 0;

static int check_device(int* sm_count)
{
    int dev = 0;
    CLUSCO_CUDA_TRY(cudaGetDevice(&dev));
    int major = 0, sms = 0;
    CLUSCO_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CLUSCO_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) return CLUSCO_ERR_UNSUPPORTED_DEVICE;
    if (sm_count) *sm_count = sms;
    return CLUSCO_OK;
}

static inline bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

__global__ void fill_kernel(float* out, size_t n, float v)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = v;
}
}  // namespace clusco

using namespace clusco;

extern "C" {

const char* clusco_status_string(int status)
{
    switch (status) {
        case CLUSCO_OK: return "ok";
        case CLUSCO_ERR_INVALID_ARG: return "invalid argument";
        case CLUSCO_ERR_WORKSPACE_TOO_SMALL: return "workspace too small or misaligned";
        case CLUSCO_ERR_UNSUPPORTED_DEVICE: return "unsupported device (needs compute capability 10.x)";
        case CLUSCO_ERR_CUDA: return "CUDA runtime error (see clusco_last_cuda_error)";
        default: return "unknown status";
    }
}

int clusco_last_cuda_error(void) { return g_last_cuda_error; }

const char* clusco_version(void) { return "0.1"; }

int clusco_engine_supported(int engine, int32_t L)
{
    if (L < 1) return 0;
    if (engine == CLUSCO_ENGINE_AUTO || engine == CLUSCO_ENGINE_FFMA) return 1;
    if (engine == CLUSCO_ENGINE_I8TC) return i8tc_supported(L) ? 1 : 0;
    return 0;
}

int clusco_i8tc_geometry(int64_t N, int32_t L, int64_t* out5)
{
    if (N < 0 || L < 1 || !out5 || !i8tc_supported(L)) return CLUSCO_ERR_INVALID_ARG;
    const Workspace w = workspace_layout(N, L);
    I8Tiles t;
    t.Tc = w.col_tiles;
    t.I_lo = 0;
    t.I_hi = w.row_tiles;
    out5[0] = N < 2 ? 0 : i8_tiles_before(t, t.I_hi);
    out5[1] = w.Lp32 / 32;
    out5[2] = 6 * 3 * I8_COL_MODELS;                         // six digit products x (3 components x column models)
    out5[3] = I8_ROW_MODELS;
    out5[4] = I8_COL_MODELS;
    return CLUSCO_OK;
}

int clusco_center(const float* coords, int64_t N, int32_t L, float* centred, float* r2, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!coords) return CLUSCO_ERR_INVALID_ARG;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    // strip per warp: the model's 3 L floats plus the alignment lead, rounded to 16 bytes
    const int64_t strip_floats = round_up(3 * (int64_t)L + 8, 4);
    if (strip_floats <= CENTER_MAX_FLOATS) {
        const int64_t blocks = (N + CENTER_WARPS - 1) / CENTER_WARPS;
        if (blocks > 0x7fffffff) return CLUSCO_ERR_INVALID_ARG;
        const size_t smem = (size_t)CENTER_WARPS * strip_floats * sizeof(float);
        CLUSCO_CUDA_TRY(cudaFuncSetAttribute(center_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        center_kernel<<<(unsigned)blocks, CENTER_WARPS * 32, smem, (cudaStream_t)stream>>>(coords, N, L, (int32_t)strip_floats,
                                                                                         centred, r2);
    } else {
        const int wpb = 8;
        const int64_t blocks = (N + wpb - 1) / wpb;
        if (blocks > 0x7fffffff) return CLUSCO_ERR_INVALID_ARG;
        center_long_kernel<<<(unsigned)blocks, wpb * 32, 0, (cudaStream_t)stream>>>(coords, N, L, centred, r2);
    }
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

size_t clusco_crmsd_allpairs_workspace(int64_t N, int32_t L)
{
    if (N < 0 || L < 1) return 0;
    if (N < 2) return 256;
    return workspace_layout(N, L).total;
}

int clusco_partition_rows(int64_t N, int32_t parts, int64_t* b)
{
    if (N < 0 || parts < 1 || !b) return CLUSCO_ERR_INVALID_ARG;
    // rows [0, r) own f(r) = r(2N - r - 1)/2 pairs; cut at equal shares, rounded to multiples of 128
    const double total = (double)N * (double)(N - 1) * 0.5;
    b[0] = 0;
    for (int32_t r = 1; r < parts; ++r) {
        const double target = total * (double)r / (double)parts;
        const double A = 2.0 * (double)N - 1.0;
        double x = (A - sqrt(fmax(0.0, A * A - 8.0 * target))) * 0.5;
        int64_t v = (int64_t)llround(x / 128.0) * 128;
        if (v < b[r - 1]) v = b[r - 1];
        if (v > N) v = N;
        b[r] = v;
    }
    b[parts] = N;
    return CLUSCO_OK;
}

static int resolve_engine(int engine, int32_t L)
{
    if (engine == CLUSCO_ENGINE_AUTO) return i8tc_supported(L) ? CLUSCO_ENGINE_I8TC : CLUSCO_ENGINE_FFMA;
    if (engine == CLUSCO_ENGINE_I8TC && !i8tc_supported(L)) return -1;
    if (engine != CLUSCO_ENGINE_FFMA && engine != CLUSCO_ENGINE_I8TC) return -1;
    return engine;
}

int clusco_allpairs_prepare(const float* coords, int64_t N, int32_t L, void* workspace, size_t workspace_bytes,
                            int engine, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    engine = resolve_engine(engine, L);
    if (engine < 0) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return CLUSCO_OK;
    if (!coords || !aligned16(coords)) return CLUSCO_ERR_INVALID_ARG;
    if (N > (int64_t)1 << 24) return CLUSCO_ERR_INVALID_ARG;
    const Workspace w = workspace_layout(N, L);
    if (!workspace || workspace_bytes < w.total || ((uintptr_t)workspace & 255u)) return CLUSCO_ERR_WORKSPACE_TOO_SMALL;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    char* ws = (char*)workspace;
    if (engine == CLUSCO_ENGINE_I8TC) return i8tc_prepare(coords, N, L, w, ws, s);   // a1 + a2 + operand planes, one launch
    ModelStat* stats = (ModelStat*)(ws + w.off_stats);
    // a1 + a2: centroid, scale exponent, sum of squares per model
    model_stats_kernel<<<(unsigned)((w.Np + 7) / 8), 256, 0, s>>>(coords, N, w.Np, L, stats);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    float* Yt = (float*)(ws + w.off_ffma);
    dim3 g((unsigned)(w.Np / 32), (unsigned)((w.Lp16 + 63) / 64));
    ffma_plane_kernel<<<g, 256, 0, s>>>(coords, N, w.Np, L, w.Lp16, stats, Yt);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

}  // extern "C"

// steps a3-a5 for rows [row_begin, row_end) from a prepared workspace; MODE selects the epilogue's sink
template <int MODE>
static int allpairs_compute_mode(int64_t N, int32_t L, int64_t row_begin, int64_t row_end, float* out_rows, const Sink& sink,
                                 void* workspace, size_t workspace_bytes, int engine, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    engine = resolve_engine(engine, L);
    if (engine < 0) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return (row_begin == 0 && row_end >= 0) ? CLUSCO_OK : CLUSCO_ERR_INVALID_ARG;
    if (row_begin < 0 || row_end < row_begin || row_end > N) return CLUSCO_ERR_INVALID_ARG;
    if (row_begin == row_end) return CLUSCO_OK;
    if (row_begin % 128 != 0 || (MODE == SINK_STORE && !out_rows)) return CLUSCO_ERR_INVALID_ARG;
    const Workspace w = workspace_layout(N, L);
    if (!workspace || workspace_bytes < w.total || ((uintptr_t)workspace & 255u)) return CLUSCO_ERR_WORKSPACE_TOO_SMALL;
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    char* ws = (char*)workspace;
    if (engine == CLUSCO_ENGINE_FFMA) {
        const ModelStat* stats = (const ModelStat*)(ws + w.off_stats);
        const float invL = 1.0f / (float)L;
        const float* Yt = (const float*)(ws + w.off_ffma);
        TileRange tr;
        tr.T = (N + FF_TILE - 1) / FF_TILE;
        tr.I_lo = row_begin / FF_TILE;
        tr.I_hi = (row_end + FF_TILE - 1) / FF_TILE;
        const int64_t W = tr.T - tr.I_lo, R = tr.I_hi - tr.I_lo;
        const int64_t tiles = R * W - R * (R - 1) / 2;
        if (tiles > 0x7fffffff) return CLUSCO_ERR_INVALID_ARG;
        gram_ffma_kernel<MODE><<<(unsigned)tiles, 256, 0, s>>>(Yt, stats, N, w.Np, w.Lp16, invL, tr, row_begin, row_end,
                                                              out_rows, sink);
        CLUSCO_CUDA_TRY(cudaGetLastError());
        return CLUSCO_OK;
    }
    return i8tc_compute<MODE>(N, L, row_begin, row_end, out_rows, sink, w, ws, sms, s);
}

extern "C" {

int clusco_allpairs_compute(int64_t N, int32_t L, int64_t row_begin, int64_t row_end, float* out_rows,
                            void* workspace, size_t workspace_bytes, int engine, void* stream)
{
    return allpairs_compute_mode<SINK_STORE>(N, L, row_begin, row_end, out_rows, Sink{}, workspace, workspace_bytes, engine,
                                             stream);
}

// NEXT-1a: threshold filter + compaction fused into the epilogue
int clusco_crmsd_allpairs_below(const float* coords, int64_t N, int32_t L, float cutoff, int64_t capacity,
                                int32_t* pair_i, int32_t* pair_j, float* pair_c, unsigned long long* count,
                                void* workspace, size_t workspace_bytes, void* stream)
{
    if (N < 0 || L < 1 || capacity < 0 || !count) return CLUSCO_ERR_INVALID_ARG;
    if (capacity > 0 && (!pair_i || !pair_j || !pair_c)) return CLUSCO_ERR_INVALID_ARG;
    if (N >= 2) {                                               // validate before touching `count`
        int st = clusco_allpairs_prepare(coords, N, L, workspace, workspace_bytes, CLUSCO_ENGINE_AUTO, stream);
        if (st != CLUSCO_OK) return st;
    } else {
        int st = check_device(nullptr);
        if (st != CLUSCO_OK) return st;
    }
    CLUSCO_CUDA_TRY(cudaMemsetAsync(count, 0, sizeof(unsigned long long), (cudaStream_t)stream));
    if (N < 2) return CLUSCO_OK;
    Sink sink{};
    sink.cutoff = cutoff;
    sink.capacity = capacity;
    sink.pair_i = pair_i;
    sink.pair_j = pair_j;
    sink.pair_c = pair_c;
    sink.count = count;
    return allpairs_compute_mode<SINK_BELOW>(N, L, 0, N, nullptr, sink, workspace, workspace_bytes, CLUSCO_ENGINE_AUTO,
                                             stream);
}

// NEXT-1b: per-model row sums and neighbour counts fused into the epilogue
int clusco_crmsd_rowstats(const float* coords, int64_t N, int32_t L, float cutoff, double* rowsum, int32_t* below,
                          void* workspace, size_t workspace_bytes, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!rowsum || !below) return CLUSCO_ERR_INVALID_ARG;
    if (N >= 2) {
        int st = clusco_allpairs_prepare(coords, N, L, workspace, workspace_bytes, CLUSCO_ENGINE_AUTO, stream);
        if (st != CLUSCO_OK) return st;
    } else {
        int st = check_device(nullptr);
        if (st != CLUSCO_OK) return st;
    }
    CLUSCO_CUDA_TRY(cudaMemsetAsync(rowsum, 0, sizeof(double) * (size_t)N, (cudaStream_t)stream));
    CLUSCO_CUDA_TRY(cudaMemsetAsync(below, 0, sizeof(int32_t) * (size_t)N, (cudaStream_t)stream));
    if (N < 2) return CLUSCO_OK;
    Sink sink{};
    sink.cutoff = cutoff;
    sink.rowsum = rowsum;
    sink.below = below;
    return allpairs_compute_mode<SINK_ROWSTATS>(N, L, 0, N, nullptr, sink, workspace, workspace_bytes, CLUSCO_ENGINE_AUTO,
                                                stream);
}

int clusco_crmsd_allpairs_ex(const float* coords, int64_t N, int32_t L, int64_t row_begin, int64_t row_end,
                             float* out_rows, void* workspace, size_t workspace_bytes, int engine, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return (row_begin == 0 && row_end >= 0) ? CLUSCO_OK : CLUSCO_ERR_INVALID_ARG;
    if (row_begin < 0 || row_end < row_begin || row_end > N) return CLUSCO_ERR_INVALID_ARG;
    if (row_begin == row_end) return CLUSCO_OK;
    if (!out_rows) return CLUSCO_ERR_INVALID_ARG;
    int st = clusco_allpairs_prepare(coords, N, L, workspace, workspace_bytes, engine, stream);
    if (st != CLUSCO_OK) return st;
    return clusco_allpairs_compute(N, L, row_begin, row_end, out_rows, workspace, workspace_bytes, engine, stream);
}

int clusco_crmsd_allpairs(const float* coords, int64_t N, int32_t L, float* out, void* workspace,
                          size_t workspace_bytes, void* stream)
{
    return clusco_crmsd_allpairs_ex(coords, N, L, 0, N < 0 ? 0 : N, out, workspace, workspace_bytes,
                                    CLUSCO_ENGINE_AUTO, stream);
}

// NEXT-2: all-versus-all dRMSD (eq. 5) as one tensor-core Gram over the distance vectors
size_t clusco_drmsd_allpairs_workspace(int64_t N, int32_t L)
{
    if (N < 0 || L < 1 || L > DG_MAX_L) return 0;
    if (N < 2 || L < 2) return 256;
    return drmsd_workspace_layout(N, L).total;
}

int clusco_drmsd_allpairs(const float* coords, int64_t N, int32_t L, float* out, void* workspace, size_t workspace_bytes,
                          void* stream)
{
    if (N < 0 || L < 1 || L > DG_MAX_L) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return CLUSCO_OK;
    if (!coords || !out) return CLUSCO_ERR_INVALID_ARG;
    if (N > (int64_t)1 << 24) return CLUSCO_ERR_INVALID_ARG;
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    if (L < 2) {                                                // a single atom has no distance: every dRMSD is 0
        CLUSCO_CUDA_TRY(cudaMemsetAsync(out, 0, sizeof(float) * (size_t)(N * (N - 1) / 2), s));
        return CLUSCO_OK;
    }
    const DWorkspace w = drmsd_workspace_layout(N, L);
    if (!workspace || workspace_bytes < w.total || ((uintptr_t)workspace & 255u)) return CLUSCO_ERR_WORKSPACE_TOO_SMALL;
    return drmsd_launch<3>(coords, N, L, 0.0, out, (char*)workspace, sms, s);
}

// NEXT-3: all-versus-all contact-map overlap (eq. 6-7) as a 0/1 int8 Gram on the same kernels
size_t clusco_cmo_allpairs_workspace(int64_t N, int32_t L)
{
    if (N < 0 || L < 1 || L > DG_MAX_L) return 0;
    if (N < 2 || L < 2) return 256;
    return drmsd_workspace_layout(N, L, 1).total;
}

int clusco_cmo_allpairs(const float* coords, int64_t N, int32_t L, float cutoff, float* out, void* workspace,
                        size_t workspace_bytes, void* stream)
{
    if (N < 0 || L < 1 || L > DG_MAX_L || !(cutoff >= 0.0f)) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return CLUSCO_OK;
    if (!coords || !out) return CLUSCO_ERR_INVALID_ARG;
    if (N > (int64_t)1 << 24) return CLUSCO_ERR_INVALID_ARG;
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    if (L < 2) {                                                // no atom pair: two empty maps, S = 100 (header)
        const size_t n = (size_t)(N * (N - 1) / 2);
        fill_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(out, n, 100.0f);
        CLUSCO_CUDA_TRY(cudaGetLastError());
        return CLUSCO_OK;
    }
    const DWorkspace w = drmsd_workspace_layout(N, L, 1);
    if (!workspace || workspace_bytes < w.total || ((uintptr_t)workspace & 255u)) return CLUSCO_ERR_WORKSPACE_TOO_SMALL;
    return drmsd_launch<1>(coords, N, L, (double)cutoff, out, (char*)workspace, sms, s);
}

// dRMSD and CMO of N models against one reference (the versus-reference form of eq. 5 and eq. 6-7)
static int ref_ova_common(int mode, const float* native, const float* coords, int64_t N, int32_t L, double cutoff, float* out,
                          void* stream)
{
    if (N < 0 || L < 1 || L > ROVA_MAX_L) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!native || !coords || !out) return CLUSCO_ERR_INVALID_ARG;
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    return mode == 0 ? ref_one_vs_all_launch<0>(native, coords, N, L, cutoff, out, sms, (cudaStream_t)stream)
                     : ref_one_vs_all_launch<1>(native, coords, N, L, cutoff, out, sms, (cudaStream_t)stream);
}

int clusco_drmsd_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float* out, void* stream)
{
    return ref_ova_common(0, native, coords, N, L, 0.0, out, stream);
}

int clusco_cmo_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float cutoff, float* out,
                          void* stream)
{
    if (!(cutoff >= 0.0f)) return CLUSCO_ERR_INVALID_ARG;
    return ref_ova_common(1, native, coords, N, L, (double)cutoff, out, stream);
}

// NEXT-4: GDT_TS / TM-score / MaxSub (the paper's fragment-seeded search, FP64): versus a reference, and all-versus-all
}  // extern "C"

template <bool ALLPAIRS>
static int gdt_launch(const float* native, const float* coords, int64_t N, int32_t L, float* out, void* stream)
{
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    const size_t smem = (size_t)(ALLPAIRS ? 2 * GDT_WARPS : 1 + GDT_WARPS) * 3 * (size_t)L * sizeof(double);
    CLUSCO_CUDA_TRY(cudaFuncSetAttribute(gdt_kernel<ALLPAIRS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1;
    CLUSCO_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gdt_kernel<ALLPAIRS>, GDT_WARPS * 32, smem));
    if (per_sm < 1) per_sm = 1;
    const int64_t units = ALLPAIRS ? N * (N - 1) / 2 : N;
    int64_t grid = (units + GDT_WARPS - 1) / GDT_WARPS;
    const int64_t cap = (int64_t)sms * per_sm;
    if (grid > cap) grid = cap;
    gdt_kernel<ALLPAIRS><<<(unsigned)grid, GDT_WARPS * 32, smem, (cudaStream_t)stream>>>(native, coords, N, L, out);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

extern "C" {

int clusco_gdt_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float* out, void* stream)
{
    if (N < 0 || L < 3 || L > GDT_MAX_L) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!native || !coords || !out) return CLUSCO_ERR_INVALID_ARG;
    return gdt_launch<false>(native, coords, N, L, out, stream);
}

int clusco_gdt_allpairs(const float* coords, int64_t N, int32_t L, float* out, void* stream)
{
    if (N < 0 || L < 3 || L > GDT_MAX_L || N > (int64_t)1 << 24) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return CLUSCO_OK;
    if (!coords || !out) return CLUSCO_ERR_INVALID_ARG;
    return gdt_launch<true>(nullptr, coords, N, L, out, stream);
}

// one launch, no scratch: every CTA centres the native into its own shared memory
int clusco_crmsd_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float* out, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!native || !coords || !out) return CLUSCO_ERR_INVALID_ARG;
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t nat_bytes = (size_t)L * sizeof(float4);
    if (nat_bytes > 200 * 1024) return CLUSCO_ERR_INVALID_ARG;        // L <= 12800 atoms
    if (!aligned16(coords)) return CLUSCO_ERR_INVALID_ARG;
    const int64_t n_blocks32 = (N + 31) / 32;
    int warps = 0, stages = 0;
    if (ova_stream_config(L, &warps, &stages)) {
        // streaming kernel: one persistent CTA per SM, every warp walks batches of 32 models
        const size_t smem = ova_stream_smem(L, warps, stages);
        int64_t grid = (n_blocks32 + warps - 1) / warps;
        if (grid > sms) grid = sms;
        const int vec = (L % 4 == 0) ? 4 : (L % 2 == 0 ? 2 : 1);
#define OVA_LAUNCH(V)                                                                                                  \
    do {                                                                                                               \
        CLUSCO_CUDA_TRY(cudaFuncSetAttribute(one_vs_all_stream_kernel<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                             (int)smem));                                                              \
        one_vs_all_stream_kernel<V><<<(unsigned)grid, warps * 32, smem, s>>>(native, coords, N, L, 1.0f / (float)L,    \
                                                                             stages, out);                             \
    } while (0)
        if (vec == 4) OVA_LAUNCH(4); else if (vec == 2) OVA_LAUNCH(2); else OVA_LAUNCH(1);
#undef OVA_LAUNCH
    } else {
        CLUSCO_CUDA_TRY(cudaFuncSetAttribute(one_vs_all_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)nat_bytes));
        int64_t grid = (n_blocks32 + OVA_WARPS - 1) / OVA_WARPS;
        const int64_t cap = (int64_t)sms * 4;
        if (grid > cap) grid = cap;
        one_vs_all_kernel<<<(unsigned)grid, OVA_WARPS * 32, nat_bytes, s>>>(native, coords, N, L, 1.0f / (float)L, out);
    }
    CLUSCO_CUDA_TRY(cudaGetLastError());
    return CLUSCO_OK;
}

// ---- host-buffer calls ---------------------------------------------------------------------------------
// Device scratch comes from a library-owned stream-ordered memory pool (one per device, kept between calls so
// that repeated calls pay no allocation; clusco_host_release() returns it to the driver), and the transfers
// run on their own stream, overlapped with the kernels chunk by chunk.
namespace {
struct HostCtx {
    cudaMemPool_t pool = nullptr;
    cudaStream_t compute = nullptr, copy = nullptr;
};
std::mutex g_host_mu;
HostCtx g_host[64];

// the caller holds g_host_mu (and keeps it for the whole host call, so that clusco_host_release() cannot destroy the
// pool and the streams under a running call)
int host_ctx_locked(HostCtx** out)
{
    int dev = 0;
    CLUSCO_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return CLUSCO_ERR_INVALID_ARG;
    HostCtx& c = g_host[dev];
    if (!c.pool) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        CLUSCO_CUDA_TRY(cudaMemPoolCreate(&c.pool, &props));
        uint64_t keep = UINT64_MAX;                          // keep freed blocks for the next call
        CLUSCO_CUDA_TRY(cudaMemPoolSetAttribute(c.pool, cudaMemPoolAttrReleaseThreshold, &keep));
        CLUSCO_CUDA_TRY(cudaStreamCreateWithFlags(&c.compute, cudaStreamNonBlocking));
        CLUSCO_CUDA_TRY(cudaStreamCreateWithFlags(&c.copy, cudaStreamNonBlocking));
    }
    *out = &c;
    return CLUSCO_OK;
}

// first error wins; later CUDA calls are still made so that every stream is drained before returning
struct ErrLatch {
    int st = CLUSCO_OK;
    void cuda(cudaError_t e)
    {
        if (e != cudaSuccess && st == CLUSCO_OK) {
            g_last_cuda_error = (int)e;
            st = CLUSCO_ERR_CUDA;
        }
    }
    void status(int s)
    {
        if (s != CLUSCO_OK && st == CLUSCO_OK) st = s;
    }
    bool ok() const { return st == CLUSCO_OK; }
};
}  // namespace

int clusco_host_release(void)
{
    std::lock_guard<std::mutex> lock(g_host_mu);
    int st = CLUSCO_OK;
    for (HostCtx& c : g_host) {
        if (!c.pool) continue;
        cudaStreamSynchronize(c.compute);
        cudaStreamSynchronize(c.copy);
        cudaStreamDestroy(c.compute);
        cudaStreamDestroy(c.copy);
        if (cudaMemPoolDestroy(c.pool) != cudaSuccess) st = CLUSCO_ERR_CUDA;
        c = HostCtx();
    }
    return st;
}

int clusco_crmsd_allpairs_host(const float* coords_host, int64_t N, int32_t L, float* out_host)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return CLUSCO_OK;
    if (!coords_host || !out_host) return CLUSCO_ERR_INVALID_ARG;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    std::lock_guard<std::mutex> lock(g_host_mu);             // one host call at a time per process
    HostCtx* ctx = nullptr;
    st = host_ctx_locked(&ctx);
    if (st != CLUSCO_OK) return st;
    const size_t in_bytes = (size_t)N * L * 3 * sizeof(float);
    const size_t n_pairs = (size_t)N * (size_t)(N - 1) / 2;
    const size_t ws_bytes = clusco_crmsd_allpairs_workspace(N, L);
    cudaStream_t sc = ctx->compute, sx = ctx->copy;
    float *d_in = nullptr, *d_out = nullptr;
    void* d_ws = nullptr;
    ErrLatch err;
    err.cuda(cudaMallocFromPoolAsync((void**)&d_in, in_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync((void**)&d_out, n_pairs * sizeof(float), ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync(&d_ws, ws_bytes, ctx->pool, sc));
    // rows are cut into chunks of equal pair count; chunk k is copied back while chunk k+1 is computed
    constexpr int MAX_CHUNKS = 8;
    int64_t bounds[MAX_CHUNKS + 1];
    const int chunks = n_pairs * sizeof(float) >= ((size_t)8 << 20) ? MAX_CHUNKS : 1;
    err.status(clusco_partition_rows(N, chunks, bounds));
    cudaEvent_t ev[MAX_CHUNKS];
    int n_ev = 0;
    if (err.ok()) {
        err.cuda(cudaMemcpyAsync(d_in, coords_host, in_bytes, cudaMemcpyHostToDevice, sc));
        err.status(clusco_allpairs_prepare(d_in, N, L, d_ws, ws_bytes, CLUSCO_ENGINE_AUTO, (void*)sc));
    }
    for (int k = 0; k < chunks && err.ok(); ++k) {
        const int64_t lo = bounds[k], hi = bounds[k + 1];
        if (hi <= lo) continue;
        const int64_t off = packed_index(lo, lo + 1, N);
        const int64_t end = hi >= N ? (int64_t)n_pairs : packed_index(hi, hi + 1, N);
        if (end <= off) continue;
        err.status(clusco_allpairs_compute(N, L, lo, hi, d_out + off, d_ws, ws_bytes, CLUSCO_ENGINE_AUTO, (void*)sc));
        if (!err.ok()) break;
        err.cuda(cudaEventCreateWithFlags(&ev[n_ev], cudaEventDisableTiming));
        if (!err.ok()) break;
        ++n_ev;
        err.cuda(cudaEventRecord(ev[n_ev - 1], sc));
        err.cuda(cudaStreamWaitEvent(sx, ev[n_ev - 1], 0));
        err.cuda(cudaMemcpyAsync(out_host + off, d_out + off, (size_t)(end - off) * sizeof(float),
                                 cudaMemcpyDeviceToHost, sx));
    }
    err.cuda(cudaStreamSynchronize(sx));
    err.cuda(cudaStreamSynchronize(sc));
    for (int k = 0; k < n_ev; ++k) cudaEventDestroy(ev[k]);
    if (d_in) cudaFreeAsync(d_in, sc);
    if (d_out) cudaFreeAsync(d_out, sc);
    if (d_ws) cudaFreeAsync(d_ws, sc);
    return err.st;
}

int clusco_crmsd_one_vs_all_host(const float* native_host, const float* coords_host, int64_t N, int32_t L,
                                 float* out_host)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!native_host || !coords_host || !out_host) return CLUSCO_ERR_INVALID_ARG;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    std::lock_guard<std::mutex> lock(g_host_mu);
    HostCtx* ctx = nullptr;
    st = host_ctx_locked(&ctx);
    if (st != CLUSCO_OK) return st;
    const size_t model_bytes = (size_t)L * 3 * sizeof(float);
    cudaStream_t sc = ctx->compute, sx = ctx->copy;
    float *d_in = nullptr, *d_nat = nullptr, *d_out = nullptr;
    ErrLatch err;
    err.cuda(cudaMallocFromPoolAsync((void**)&d_in, (size_t)N * model_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync((void**)&d_nat, model_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync((void**)&d_out, (size_t)N * sizeof(float), ctx->pool, sc));
    // the models go up in chunks (a multiple of 32 models, about 64 MB) on the copy stream; each chunk is
    // scored as soon as it has landed, so the kernels hide behind the transfer
    int64_t per = ((int64_t)(64 << 20) / (int64_t)model_bytes) / 32 * 32;
    if (per < 32) per = 32;
    const int64_t chunks = (N + per - 1) / per;
    cudaEvent_t ready = nullptr, alloc_done = nullptr;
    err.cuda(cudaEventCreateWithFlags(&ready, cudaEventDisableTiming));
    err.cuda(cudaEventCreateWithFlags(&alloc_done, cudaEventDisableTiming));
    if (err.ok()) {
        err.cuda(cudaMemcpyAsync(d_nat, native_host, model_bytes, cudaMemcpyHostToDevice, sc));
        err.cuda(cudaEventRecord(alloc_done, sc));                    // the pool blocks are ordered on sc
        err.cuda(cudaStreamWaitEvent(sx, alloc_done, 0));
    }
    for (int64_t k = 0; k < chunks && err.ok(); ++k) {
        const int64_t m0 = k * per, cnt = (m0 + per <= N ? per : N - m0);
        err.cuda(cudaMemcpyAsync(d_in + m0 * (int64_t)L * 3, coords_host + m0 * (int64_t)L * 3, (size_t)cnt * model_bytes,
                                 cudaMemcpyHostToDevice, sx));
        err.cuda(cudaEventRecord(ready, sx));
        err.cuda(cudaStreamWaitEvent(sc, ready, 0));
        err.status(clusco_crmsd_one_vs_all(d_nat, d_in + m0 * (int64_t)L * 3, cnt, L, d_out + m0, (void*)sc));
    }
    if (err.ok()) err.cuda(cudaMemcpyAsync(out_host, d_out, (size_t)N * sizeof(float), cudaMemcpyDeviceToHost, sc));
    err.cuda(cudaStreamSynchronize(sx));
    err.cuda(cudaStreamSynchronize(sc));
    if (ready) cudaEventDestroy(ready);
    if (alloc_done) cudaEventDestroy(alloc_done);
    if (d_in) cudaFreeAsync(d_in, sc);
    if (d_nat) cudaFreeAsync(d_nat, sc);
    if (d_out) cudaFreeAsync(d_out, sc);
    return err.st;
}

// ---- host-buffer forms of the fused consumers: the coordinates go up, only the triples / the
// per-model statistics come down -- 18 MB instead of the 200 MB matrix at C3 ---------------------------------------
int clusco_crmsd_allpairs_below_host(const float* coords_host, int64_t N, int32_t L, float cutoff, int64_t capacity,
                                     int32_t* pair_i_host, int32_t* pair_j_host, float* pair_c_host,
                                     unsigned long long* count_host)
{
    if (N < 0 || L < 1 || capacity < 0 || !count_host) return CLUSCO_ERR_INVALID_ARG;
    if (capacity > 0 && (!pair_i_host || !pair_j_host || !pair_c_host)) return CLUSCO_ERR_INVALID_ARG;
    *count_host = 0ull;
    if (N < 2) return CLUSCO_OK;
    if (!coords_host) return CLUSCO_ERR_INVALID_ARG;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    std::lock_guard<std::mutex> lock(g_host_mu);
    HostCtx* ctx = nullptr;
    st = host_ctx_locked(&ctx);
    if (st != CLUSCO_OK) return st;
    const size_t in_bytes = (size_t)N * L * 3 * sizeof(float);
    const size_t ws_bytes = clusco_crmsd_allpairs_workspace(N, L);
    const int64_t n_pairs = N * (N - 1) / 2;
    cudaStream_t sc = ctx->compute;
    float* d_in = nullptr;
    void* d_ws = nullptr;
    unsigned long long* d_count = nullptr;
    char* d_tri = nullptr;                                   // [pair_i | pair_j | pair_c], dev_cap entries each
    ErrLatch err;
    err.cuda(cudaMallocFromPoolAsync((void**)&d_in, in_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync(&d_ws, ws_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync((void**)&d_count, sizeof(unsigned long long), ctx->pool, sc));
    // the caller's capacity may be a worst-case bound (all N(N-1)/2 pairs); the device staging starts at 4 Mi triples
    // and a second pass of the compute stage follows only if the count says more are wanted AND the caller has room
    int64_t dev_cap = capacity < n_pairs ? capacity : n_pairs;
    if (dev_cap > ((int64_t)1 << 22)) dev_cap = (int64_t)1 << 22;
    unsigned long long found = 0ull;
    if (err.ok()) err.cuda(cudaMemcpyAsync(d_in, coords_host, in_bytes, cudaMemcpyHostToDevice, sc));
    for (int pass = 0; pass < 2 && err.ok(); ++pass) {
        if (dev_cap > 0) err.cuda(cudaMallocFromPoolAsync((void**)&d_tri, (size_t)dev_cap * 12, ctx->pool, sc));
        if (!err.ok()) break;
        int32_t* d_i = (int32_t*)d_tri;
        int32_t* d_j = d_i + dev_cap;
        float* d_c = (float*)(d_j + dev_cap);
        if (pass == 0) {
            err.status(clusco_crmsd_allpairs_below(d_in, N, L, cutoff, dev_cap, d_i, d_j, d_c, d_count, d_ws, ws_bytes,
                                                   (void*)sc));
        } else {                                             // the workspace is still prepared: compute stage only
            err.cuda(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), sc));
            Sink sink{};
            sink.cutoff = cutoff;
            sink.capacity = dev_cap;
            sink.pair_i = d_i;
            sink.pair_j = d_j;
            sink.pair_c = d_c;
            sink.count = d_count;
            err.status(allpairs_compute_mode<SINK_BELOW>(N, L, 0, N, nullptr, sink, d_ws, ws_bytes, CLUSCO_ENGINE_AUTO,
                                                         (void*)sc));
        }
        if (!err.ok()) break;
        err.cuda(cudaMemcpyAsync(&found, d_count, sizeof(found), cudaMemcpyDeviceToHost, sc));
        err.cuda(cudaStreamSynchronize(sc));
        if (!err.ok()) break;
        const int64_t want = (int64_t)found < capacity ? (int64_t)found : capacity;
        if (want <= dev_cap) {
            if (want > 0) {
                err.cuda(cudaMemcpyAsync(pair_i_host, d_i, (size_t)want * 4, cudaMemcpyDeviceToHost, sc));
                err.cuda(cudaMemcpyAsync(pair_j_host, d_j, (size_t)want * 4, cudaMemcpyDeviceToHost, sc));
                err.cuda(cudaMemcpyAsync(pair_c_host, d_c, (size_t)want * 4, cudaMemcpyDeviceToHost, sc));
            }
            break;
        }
        cudaFreeAsync(d_tri, sc);                            // more wanted than staged: once more with room for all
        d_tri = nullptr;
        dev_cap = want;
    }
    err.cuda(cudaStreamSynchronize(sc));
    if (err.ok()) *count_host = found;
    if (d_tri) cudaFreeAsync(d_tri, sc);
    if (d_count) cudaFreeAsync(d_count, sc);
    if (d_in) cudaFreeAsync(d_in, sc);
    if (d_ws) cudaFreeAsync(d_ws, sc);
    return err.st;
}

int clusco_crmsd_rowstats_host(const float* coords_host, int64_t N, int32_t L, float cutoff, double* rowsum_host,
                               int32_t* below_host)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!coords_host || !rowsum_host || !below_host) return CLUSCO_ERR_INVALID_ARG;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    std::lock_guard<std::mutex> lock(g_host_mu);
    HostCtx* ctx = nullptr;
    st = host_ctx_locked(&ctx);
    if (st != CLUSCO_OK) return st;
    const size_t in_bytes = (size_t)N * L * 3 * sizeof(float);
    const size_t ws_bytes = clusco_crmsd_allpairs_workspace(N, L);
    cudaStream_t sc = ctx->compute;
    float* d_in = nullptr;
    void* d_ws = nullptr;
    double* d_sum = nullptr;
    int32_t* d_below = nullptr;
    ErrLatch err;
    err.cuda(cudaMallocFromPoolAsync((void**)&d_in, in_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync(&d_ws, ws_bytes, ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync((void**)&d_sum, (size_t)N * sizeof(double), ctx->pool, sc));
    err.cuda(cudaMallocFromPoolAsync((void**)&d_below, (size_t)N * sizeof(int32_t), ctx->pool, sc));
    if (err.ok()) {
        err.cuda(cudaMemcpyAsync(d_in, coords_host, in_bytes, cudaMemcpyHostToDevice, sc));
        err.status(clusco_crmsd_rowstats(d_in, N, L, cutoff, d_sum, d_below, d_ws, ws_bytes, (void*)sc));
    }
    if (err.ok()) {
        err.cuda(cudaMemcpyAsync(rowsum_host, d_sum, (size_t)N * sizeof(double), cudaMemcpyDeviceToHost, sc));
        err.cuda(cudaMemcpyAsync(below_host, d_below, (size_t)N * sizeof(int32_t), cudaMemcpyDeviceToHost, sc));
    }
    err.cuda(cudaStreamSynchronize(sc));
    if (d_in) cudaFreeAsync(d_in, sc);
    if (d_ws) cudaFreeAsync(d_ws, sc);
    if (d_sum) cudaFreeAsync(d_sum, sc);
    if (d_below) cudaFreeAsync(d_below, sc);
    return err.st;
}

}  // extern "C"
