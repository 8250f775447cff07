// i8_layout.cuh -- operand-image layout of the tensor-core engine (gram_i8tc.cuh), host- and device-callable: where a
// (model, component, digit, atom) byte sits in the A and B images that i8_prep_kernel writes and the MMAs of
// gram_i8tc_kernel read.  No PTX and no arithmetic of the method beyond the digit split, so that a host program can build
// the images with the very functions the kernel uses (tests/i8_layout_harness.cu) and check them against a model of the
// MMA sequence without a GPU.
#pragma once
#include "common.cuh"

namespace clusco {

// byte offset of K slot k of row `row` inside a slab (tcgen05's canonical K-major, no-swizzle core matrices: 8 rows x 16
// bytes each, 256 bytes per 8-row group, the two 16-byte K halves of a row group 128 bytes apart)
__host__ __device__ constexpr int i8_slab_offset(int row, int k) { return (row >> 3) * 256 + (k >> 4) * 128 + (row & 7) * 16 + (k & 15); }
// slab index of (digit a, k-step k) inside a row tile's A image: Ap[row_tile][digit][kstep][I8_A_SLAB]
__host__ __device__ constexpr int i8_a_slab_index(int a, int k, int ks) { return a * ks + k; }

// position of column model m16 (0..15) of a tile among the 16 B rows of a component block, and of its epilogue record
__host__ __device__ __forceinline__ int i8_col_slot(int m16) { return (m16 & 8) | ((m16 & 3) << 1) | ((m16 >> 2) & 1); }
__host__ __device__ __forceinline__ int i8_stat_slot(int m16) { return ((m16 & 3) << 2) | ((m16 >> 2) & 3); }

// I = d0 2^16 + d1 2^8 + d2 with signed 8-bit digits (|I| <= 127/128 2^23, so d0 fits too)
__host__ __device__ __forceinline__ void i8_digits(int I, int& d0, int& d1, int& d2)
{
    d2 = (int)(int8_t)(I & 0xff);
    const int I1 = (I - d2) >> 8;
    d1 = (int)(int8_t)(I1 & 0xff);
    d0 = (I1 - d1) >> 8;
}

// The stores of one packing lane: model slot n, k-step kk of ks, lane j (atoms and K slots 4 j .. 4 j + 3 of the k-step),
// row group p (component 0..2, or 3 = the zero rows of the A image), with w0, w1, w2 the digit words (digit g of the lane's
// four atoms, one byte each) -- into the A image (row tile n / 32: TMEM lane 32 w + 8 p + r for model 8 w + r of the tile)
// and, for p < 3, into the B image (column tile n / 16: row 16 p + i8_col_slot(n % 16) of each digit block of 48 rows).
__host__ __device__ __forceinline__ void i8_store_lane_words(int8_t* Ap, int8_t* Bp, bool to_a, bool to_b, int64_t n, int ks,
                                                            int kk, int j, int p, uint32_t w0, uint32_t w1, uint32_t w2)
{
    if (to_a) {
        const int a_w = (int)(n & 31) >> 3, a_r = (int)(n & 7);
        int8_t* tile = Ap + (n >> 5) * 3 * ks * (int64_t)I8_A_SLAB + i8_slab_offset(8 * (4 * a_w + p) + a_r, 4 * j);
        *reinterpret_cast<uint32_t*>(tile + (int64_t)i8_a_slab_index(0, kk, ks) * I8_A_SLAB) = p < 3 ? w0 : 0u;
        *reinterpret_cast<uint32_t*>(tile + (int64_t)i8_a_slab_index(1, kk, ks) * I8_A_SLAB) = p < 3 ? w1 : 0u;
        *reinterpret_cast<uint32_t*>(tile + (int64_t)i8_a_slab_index(2, kk, ks) * I8_A_SLAB) = p < 3 ? w2 : 0u;
    }
    if (to_b && p < 3) {
        const int b_o = i8_col_slot((int)(n & 15));
        int8_t* slab = Bp + ((n >> 4) * ks + kk) * (int64_t)I8_B_SLAB + i8_slab_offset(16 * p + b_o, 4 * j);
        *reinterpret_cast<uint32_t*>(slab) = w0;
        *reinterpret_cast<uint32_t*>(slab + 48 * 32) = w1;
        *reinterpret_cast<uint32_t*>(slab + 96 * 32) = w2;
    }
}

}  // namespace clusco
