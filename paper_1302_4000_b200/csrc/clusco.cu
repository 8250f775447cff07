// clusco.cu -- the C ABI declared in include/clusco.h: argument validation, workspace carving and kernel
// launches.  Every step of the path runs in the kernels of this directory; there is no CPU fallback.
#include <math.h>
#include <string.h>

#include "common.cuh"
#include "epilogue.cuh"
#include "gram_ffma.cuh"
#include "gram_i8tc.cuh"
#include "one_vs_all.cuh"
#include "prep.cuh"

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

int clusco_center(const float* coords, int64_t N, int32_t L, float* centred, float* r2, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!coords) return CLUSCO_ERR_INVALID_ARG;
    int st = check_device(nullptr);
    if (st != CLUSCO_OK) return st;
    const int wpb = 8;
    const int64_t blocks = (N + wpb - 1) / wpb;
    if (blocks > 0x7fffffff) return CLUSCO_ERR_INVALID_ARG;
    center_kernel<<<(unsigned)blocks, wpb * 32, 0, (cudaStream_t)stream>>>(coords, N, L, centred, r2);
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
    ModelStat* stats = (ModelStat*)(ws + w.off_stats);
    // a1 + a2: centroid, scale exponent, sum of squares per model
    model_stats_kernel<<<(unsigned)((w.Np + 7) / 8), 256, 0, s>>>(coords, N, w.Np, L, stats);
    CLUSCO_CUDA_TRY(cudaGetLastError());
    if (engine == CLUSCO_ENGINE_FFMA) {
        float* Yt = (float*)(ws + w.off_ffma);
        dim3 g((unsigned)(w.Np / 32), (unsigned)((w.Lp16 + 63) / 64));
        ffma_plane_kernel<<<g, 256, 0, s>>>(coords, N, w.Np, L, w.Lp16, stats, Yt);
        CLUSCO_CUDA_TRY(cudaGetLastError());
        return CLUSCO_OK;
    }
    return i8tc_prepare(coords, N, L, w, ws, stats, s);
}

int clusco_allpairs_compute(int64_t N, int32_t L, int64_t row_begin, int64_t row_end, float* out_rows,
                            void* workspace, size_t workspace_bytes, int engine, void* stream)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    engine = resolve_engine(engine, L);
    if (engine < 0) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return (row_begin == 0 && row_end >= 0) ? CLUSCO_OK : CLUSCO_ERR_INVALID_ARG;
    if (row_begin < 0 || row_end < row_begin || row_end > N) return CLUSCO_ERR_INVALID_ARG;
    if (row_begin == row_end) return CLUSCO_OK;
    if (row_begin % 128 != 0 || !out_rows) return CLUSCO_ERR_INVALID_ARG;
    const Workspace w = workspace_layout(N, L);
    if (!workspace || workspace_bytes < w.total || ((uintptr_t)workspace & 255u)) return CLUSCO_ERR_WORKSPACE_TOO_SMALL;
    int sms = 0;
    int st = check_device(&sms);
    if (st != CLUSCO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    char* ws = (char*)workspace;
    ModelStat* stats = (ModelStat*)(ws + w.off_stats);
    const float invL = 1.0f / (float)L;
    if (engine == CLUSCO_ENGINE_FFMA) {
        const float* Yt = (const float*)(ws + w.off_ffma);
        TileRange tr;
        tr.T = (N + FF_TILE - 1) / FF_TILE;
        tr.I_lo = row_begin / FF_TILE;
        tr.I_hi = (row_end + FF_TILE - 1) / FF_TILE;
        const int64_t W = tr.T - tr.I_lo, R = tr.I_hi - tr.I_lo;
        const int64_t tiles = R * W - R * (R - 1) / 2;
        if (tiles > 0x7fffffff) return CLUSCO_ERR_INVALID_ARG;
        gram_ffma_kernel<<<(unsigned)tiles, 256, 0, s>>>(Yt, stats, N, w.Np, w.Lp16, invL, tr, row_begin, row_end,
                                                        out_rows);
        CLUSCO_CUDA_TRY(cudaGetLastError());
        return CLUSCO_OK;
    }
    return i8tc_compute(N, L, row_begin, row_end, out_rows, w, ws, stats, sms, s);
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

// scratch for the centred native lives in a small per-call device allocation ordered on the stream
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
    const size_t natc_sz = (size_t)round_up((int64_t)nat_bytes, 256);
    const size_t natq_sz = (size_t)round_up((int64_t)((L + 3) / 4) * OVA_NATQ_FLOATS * 4, 256);
    char* scratch = nullptr;
    CLUSCO_CUDA_TRY(cudaMallocAsync((void**)&scratch, natc_sz + natq_sz + 256, s));
    float4* natc = (float4*)scratch;
    float* natq = (float*)(scratch + natc_sz);
    NativeStat* nstat = (NativeStat*)(scratch + natc_sz + natq_sz);
    native_prep_kernel<<<1, 256, 0, s>>>(native, L, natc, natq, nstat);
    CLUSCO_CUDA_TRY(cudaGetLastError());
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
        one_vs_all_stream_kernel<V><<<(unsigned)grid, warps * 32, smem, s>>>(natq, nstat, coords, N, L,                \
                                                                             1.0f / (float)L, stages, out);            \
    } while (0)
        if (vec == 4) OVA_LAUNCH(4); else if (vec == 2) OVA_LAUNCH(2); else OVA_LAUNCH(1);
#undef OVA_LAUNCH
    } else {
        static thread_local size_t smem_set = 0;
        if (nat_bytes > 48 * 1024 && nat_bytes > smem_set) {
            CLUSCO_CUDA_TRY(cudaFuncSetAttribute(one_vs_all_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 (int)nat_bytes));
            smem_set = nat_bytes;
        }
        int64_t grid = (n_blocks32 + OVA_WARPS - 1) / OVA_WARPS;
        const int64_t cap = (int64_t)sms * 8;
        if (grid > cap) grid = cap;
        one_vs_all_kernel<<<(unsigned)grid, OVA_WARPS * 32, nat_bytes, s>>>(natc, nstat, coords, N, L,
                                                                           1.0f / (float)L, out);
    }
    CLUSCO_CUDA_TRY(cudaGetLastError());
    CLUSCO_CUDA_TRY(cudaFreeAsync(scratch, s));
    return CLUSCO_OK;
}

int clusco_crmsd_allpairs_host(const float* coords_host, int64_t N, int32_t L, float* out_host)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N < 2) return CLUSCO_OK;
    if (!coords_host || !out_host) return CLUSCO_ERR_INVALID_ARG;
    const size_t in_bytes = (size_t)N * L * 3 * sizeof(float);
    const size_t n_pairs = (size_t)N * (size_t)(N - 1) / 2;
    const size_t ws_bytes = clusco_crmsd_allpairs_workspace(N, L);
    float *d_in = nullptr, *d_out = nullptr;
    void* d_ws = nullptr;
    cudaStream_t s;
    CLUSCO_CUDA_TRY(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
    int st = CLUSCO_OK;
    cudaError_t e;
    if ((e = cudaMalloc((void**)&d_in, in_bytes)) != cudaSuccess ||
        (e = cudaMalloc((void**)&d_out, n_pairs * sizeof(float))) != cudaSuccess ||
        (e = cudaMalloc(&d_ws, ws_bytes)) != cudaSuccess) {
        g_last_cuda_error = (int)e;
        st = CLUSCO_ERR_CUDA;
    }
    if (st == CLUSCO_OK && (e = cudaMemcpyAsync(d_in, coords_host, in_bytes, cudaMemcpyHostToDevice, s)) != cudaSuccess) {
        g_last_cuda_error = (int)e;
        st = CLUSCO_ERR_CUDA;
    }
    if (st == CLUSCO_OK) st = clusco_crmsd_allpairs(d_in, N, L, d_out, d_ws, ws_bytes, (void*)s);
    if (st == CLUSCO_OK &&
        ((e = cudaMemcpyAsync(out_host, d_out, n_pairs * sizeof(float), cudaMemcpyDeviceToHost, s)) != cudaSuccess ||
         (e = cudaStreamSynchronize(s)) != cudaSuccess)) {
        g_last_cuda_error = (int)e;
        st = CLUSCO_ERR_CUDA;
    }
    cudaFree(d_in);
    cudaFree(d_out);
    cudaFree(d_ws);
    cudaStreamDestroy(s);
    return st;
}

int clusco_crmsd_one_vs_all_host(const float* native_host, const float* coords_host, int64_t N, int32_t L,
                                 float* out_host)
{
    if (N < 0 || L < 1) return CLUSCO_ERR_INVALID_ARG;
    if (N == 0) return CLUSCO_OK;
    if (!native_host || !coords_host || !out_host) return CLUSCO_ERR_INVALID_ARG;
    const size_t in_bytes = (size_t)N * L * 3 * sizeof(float), nat_bytes = (size_t)L * 3 * sizeof(float);
    float *d_in = nullptr, *d_nat = nullptr, *d_out = nullptr;
    cudaStream_t s;
    CLUSCO_CUDA_TRY(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
    int st = CLUSCO_OK;
    cudaError_t e;
    if ((e = cudaMalloc((void**)&d_in, in_bytes)) != cudaSuccess ||
        (e = cudaMalloc((void**)&d_nat, nat_bytes)) != cudaSuccess ||
        (e = cudaMalloc((void**)&d_out, (size_t)N * sizeof(float))) != cudaSuccess ||
        (e = cudaMemcpyAsync(d_nat, native_host, nat_bytes, cudaMemcpyHostToDevice, s)) != cudaSuccess ||
        (e = cudaMemcpyAsync(d_in, coords_host, in_bytes, cudaMemcpyHostToDevice, s)) != cudaSuccess) {
        g_last_cuda_error = (int)e;
        st = CLUSCO_ERR_CUDA;
    }
    if (st == CLUSCO_OK) st = clusco_crmsd_one_vs_all(d_nat, d_in, N, L, d_out, (void*)s);
    if (st == CLUSCO_OK &&
        ((e = cudaMemcpyAsync(out_host, d_out, (size_t)N * sizeof(float), cudaMemcpyDeviceToHost, s)) != cudaSuccess ||
         (e = cudaStreamSynchronize(s)) != cudaSuccess)) {
        g_last_cuda_error = (int)e;
        st = CLUSCO_ERR_CUDA;
    }
    cudaFree(d_in);
    cudaFree(d_nat);
    cudaFree(d_out);
    cudaStreamDestroy(s);
    return st;
}

}  // extern "C"
