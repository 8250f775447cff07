// i8_layout_harness.cu -- host-only check of the tensor-core engine's operand images (no GPU, no CUDA call).
//
// Builds the A and B images of a small (N, L) problem from random 24-bit fixed-point integers with the SAME functions
// i8_prep_kernel uses (paper_1302_4000_b200/csrc/i8_layout.cuh: i8_digits, i8_store_lane_words, in the
// kernel's loop structure over rounds, k-steps, packing lanes and components), then plays the MMA sequence of
// gram_i8tc_kernel over every tile on a plain model of tcgen05.mma kind::i8 with K-major no-swizzle operands
// (D[row][col] += sum_k A[row][k] B[col][k], byte (row, k) of an operand at i8_slab_offset(row, k)), and compares every
// accumulator entry with the level sums V0 = d0.d0, V1 = d0.d1 + d1.d0, V2 = d0.d2 + d1.d1 + d2.d0 taken directly from
// the integers at the place the epilogue reads it: TMEM lane 32 w + 8 p + r, column 48 v + 16 q + o.
// Also checked: every byte of the images the MMAs read is written by the prepare step (no stale workspace bytes), nothing
// is written outside them, and the zero rows (p = 3) stay zero.
//
//   usage: i8_layout_harness N L seed      -> prints "OK ..." and returns 0, or the first mismatches and returns 1
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "../paper_1302_4000_b200/csrc/i8_layout.cuh"

using namespace clusco;

static uint64_t rng_state;
static uint32_t rng()
{
    rng_state = rng_state * 6364136223846793005ull + 1442695040888963407ull;
    return (uint32_t)(rng_state >> 33);
}

int main(int argc, char** argv)
{
    if (argc < 4) return 2;
    const int64_t N = atoll(argv[1]);
    const int L = atoi(argv[2]);
    rng_state = 0x9E3779B97F4A7C15ull ^ (uint64_t)atoll(argv[3]);
    const int ks = (L + 31) / 32;
    const int SL = 3 * ks;                                       // slabs of a row tile's A image
    const int64_t Np = (N + 127) / 128 * 128;
    const int64_t row_tiles = (N + I8_ROW_MODELS - 1) / I8_ROW_MODELS, col_tiles = (N + I8_COL_MODELS - 1) / I8_COL_MODELS;
    const int64_t row_slots = row_tiles * I8_ROW_MODELS, col_slots = col_tiles * I8_COL_MODELS;
    const size_t a_bytes = (size_t)row_tiles * SL * I8_A_SLAB, b_bytes = (size_t)col_tiles * ks * I8_B_SLAB;
    const size_t guard = 4096;

    // the fixed-point integers |I| <= 127/128 2^23 (a few at the extremes), zero beyond N
    const int IMAX = (127 << 16);
    std::vector<int> I((size_t)Np * L * 3, 0);
    for (int64_t n = 0; n < N; ++n)
        for (int e = 0; e < 3 * L; ++e) {
            const uint32_t u = rng();
            int v = (int)(u % (2u * IMAX + 1u)) - IMAX;
            if ((u >> 28) == 0) v = (u & 1) ? IMAX : -IMAX;
            I[(size_t)n * L * 3 + e] = v;
        }

    // ---- the prepare step's packing, twice over differently poisoned buffers ----
    std::vector<int8_t> img[2];
    for (int pass = 0; pass < 2; ++pass) {
        img[pass].assign(a_bytes + b_bytes + 2 * guard, pass ? (int8_t)0x33 : (int8_t)0x77);
        int8_t* Ap = img[pass].data() + guard;
        int8_t* Bp = Ap + a_bytes;                               // (the guard after B is the buffer's tail)
        for (int64_t n = 0; n < Np; ++n) {
            const int n_el = n < N ? 3 * L : 0;
            for (int r = 0; r < 2; ++r) {
                if (4 * r >= ks) break;
                int strip[4 * 97];
                for (int el = 0; el < 384; ++el) strip[el + el / 96] = 384 * r + el < n_el ? I[(size_t)n * L * 3 + 384 * r + el] : 0;
                for (int lane = 0; lane < 32; ++lane) {
                    const int sub = lane >> 3, j = lane & 7, kk = 4 * r + sub;
                    if (kk >= ks) continue;
                    for (int p = 0; p < 3; ++p) {
                        uint32_t w[3] = {0u, 0u, 0u};
                        for (int i = 0; i < 4; ++i) {
                            int d0, d1, d2;
                            i8_digits(strip[97 * sub + 3 * (4 * j + i) + p], d0, d1, d2);
                            w[0] |= (uint32_t)(d0 & 0xff) << (8 * i);
                            w[1] |= (uint32_t)(d1 & 0xff) << (8 * i);
                            w[2] |= (uint32_t)(d2 & 0xff) << (8 * i);
                        }
                        i8_store_lane_words(Ap, Bp, n < row_slots, n < col_slots, n, ks, kk, j, p, w[0], w[1], w[2]);
                    }
                    i8_store_lane_words(Ap, Bp, n < row_slots, false, n, ks, kk, j, 3, 0u, 0u, 0u);
                }
            }
        }
    }
    int bad = 0;
    for (size_t k = 0; k < img[0].size() && bad < 5; ++k) {
        const bool inside = k >= guard && k < guard + a_bytes + b_bytes;
        const bool written = img[0][k] == img[1][k];
        if (inside != written) {
            printf("byte %zu (%s): %s\n", k - guard, k - guard < a_bytes ? "A image" : "B image",
                   inside ? "read by the MMAs but never written" : "written outside the images");
            ++bad;
        }
    }
    if (bad) return 1;
    const int8_t* Ap = img[0].data() + guard;
    const int8_t* Bp = Ap + a_bytes;

    // ---- digits of every model, for the direct level sums ----
    std::vector<int8_t> dg((size_t)Np * L * 3 * 3);              // [n][atom][comp][digit]
    for (size_t e = 0; e < (size_t)Np * L * 3; ++e) {
        int d0, d1, d2;
        i8_digits(I[e], d0, d1, d2);
        if (d0 < -127 || d0 > 127 || d1 < -128 || d1 > 127 || d2 < -128 || d2 > 127 || ((d0 * 256 + d1) * 256 + d2) != I[e]) {
            printf("digit split of %d is wrong: %d %d %d\n", I[e], d0, d1, d2);
            return 1;
        }
        dg[3 * e + 0] = (int8_t)d0; dg[3 * e + 1] = (int8_t)d1; dg[3 * e + 2] = (int8_t)d2;
    }

    // ---- the MMA sequence of gram_i8tc_kernel, tile by tile ----
    long long checked = 0;
    std::vector<int32_t> D(128 * 144);
    auto mma = [&](int dcol0, int ncols, const int8_t* a_slab, const int8_t* b_slab) {
        for (int row = 0; row < 128; ++row)
            for (int c = 0; c < ncols; ++c) {
                int32_t s = 0;
                for (int k = 0; k < 32; ++k) s += (int32_t)a_slab[i8_slab_offset(row, k)] * (int32_t)b_slab[i8_slab_offset(c, k)];
                D[row * 144 + dcol0 + c] += s;
            }
    };
    for (int64_t Ti = 0; Ti < row_tiles; ++Ti)
        for (int64_t Tj = 2 * Ti; Tj < col_tiles; ++Tj) {
            std::fill(D.begin(), D.end(), 0);
            const int8_t* At = Ap + (size_t)Ti * SL * I8_A_SLAB;
            const int8_t* Bt = Bp + (size_t)Tj * ks * I8_B_SLAB;
            for (int k = 0; k < ks; ++k) {                       // digit a, k-step k: slab a ks + k (TMEM column 8 (a ks + k))
                mma(0, 144, At + (size_t)(k) * I8_A_SLAB, Bt + (size_t)k * I8_B_SLAB);
                mma(48, 96, At + (size_t)(ks + k) * I8_A_SLAB, Bt + (size_t)k * I8_B_SLAB);
                mma(96, 48, At + (size_t)(2 * ks + k) * I8_A_SLAB, Bt + (size_t)k * I8_B_SLAB);
            }
            for (int w = 0; w < 4; ++w)
                for (int r = 0; r < 8; ++r) {
                    const int64_t mi = Ti * I8_ROW_MODELS + 8 * w + r;
                    for (int m = 0; m < 16; ++m) {
                        const int64_t mj = Tj * I8_COL_MODELS + m;
                        const int o = i8_col_slot(m);
                        for (int p = 0; p < 4; ++p)
                            for (int q = 0; q < 3; ++q) {
                                long long V[3] = {0, 0, 0};
                                if (p < 3)
                                    for (int at = 0; at < L; ++at) {
                                        const int8_t* a = &dg[(((size_t)mi * L + at) * 3 + p) * 3];
                                        const int8_t* b = &dg[(((size_t)mj * L + at) * 3 + q) * 3];
                                        V[0] += a[0] * b[0];
                                        V[1] += a[0] * b[1] + a[1] * b[0];
                                        V[2] += a[0] * b[2] + a[1] * b[1] + a[2] * b[0];
                                    }
                                for (int v = 0; v < 3; ++v) {
                                    const int32_t got = D[(32 * w + 8 * p + r) * 144 + 48 * v + 16 * q + o];
                                    ++checked;
                                    if ((long long)got != V[v]) {
                                        if (bad < 5)
                                            printf("tile (%lld, %lld) models (%lld, %lld) p %d q %d level %d: accumulator %d, direct %lld\n",
                                                   (long long)Ti, (long long)Tj, (long long)mi, (long long)mj, p, q, v, got, V[v]);
                                        ++bad;
                                    }
                                }
                            }
                    }
                }
        }
    if (bad) {
        printf("%d mismatches of %lld\n", bad, checked);
        return 1;
    }
    printf("OK N=%lld L=%d ksteps=%d slabs=%d entries=%lld\n", (long long)N, L, ks, SL, checked);
    return 0;
}
