"""Host-side checks of the integer bounds the tensor-core engine's exactness rests on (no GPU, no oracle,
no product code: the digit split is restated here from its definition and pushed through numpy int64 / Python integers).

The engine writes a scaled centred coordinate as a 24-bit integer I = round(a * KAPPA * 2^23), KAPPA = 127/128, |a| < 1, splits it
into signed 8-bit digits I = d0 2^16 + d1 2^8 + d2 and accumulates, per pair and matrix entry, the level sums
    V0 = sum d0 d0',  V1 = sum (d0 d1' + d1 d0'),  V2 = sum (d0 d2' + d1 d1' + d2 d0')
in int32; the epilogue forms T = 2^8 V1 + V2 in int32.  What has to hold for L <= 256 atoms (8 k-steps of 32):
  * every digit fits int8 and |d0| <= 127,
  * |V0|, |V1|, |V2| and |T| stay below 2^31 for ANY digit pattern,
  * 2^16 V0 + T equals the exact product sum up to the two dropped levels, whose size is bounded by L (2^16 + 2^14).
"""
import numpy as np

KAPPA = 127.0 / 128.0
L_MAX = 256


def split(I):
    """Signed base-256 digits of a 24-bit integer, low digits in [-128, 127] (the rounding the prepare kernel's comment states)."""
    I = np.asarray(I, dtype=np.int64)
    d2 = ((I + 128) % 256) - 128
    I1 = (I - d2) // 256
    d1 = ((I1 + 128) % 256) - 128
    d0 = (I1 - d1) // 256
    return d0, d1, d2


def test_digits_fit_int8_and_top_digit_is_bounded_by_kappa():
    edge = np.array([0, 1, -1, 127, 128, -128, -129, 32767, 32768, -32768, -32769], dtype=np.int64)
    Imax = int(np.floor(KAPPA * 2 ** 23 + 0.5))                      # |a| < 1  =>  |I| <= round(KAPPA 2^23)
    I = np.concatenate([edge, np.array([Imax, -Imax, Imax - 1, -Imax + 1]),
                        np.random.default_rng(1).integers(-Imax, Imax + 1, size=200_000)])
    d0, d1, d2 = split(I)
    assert np.array_equal(d0 * 65536 + d1 * 256 + d2, I)
    for d in (d1, d2):
        assert d.min() >= -128 and d.max() <= 127
    assert np.abs(d0).max() <= 127                                   # what KAPPA = 127/128 buys: no +128 in the top digit


def test_level_sums_and_their_combination_fit_int32_for_any_digits():
    # worst case by absolute value: every digit at its extreme, signs aligned
    d0, d1 = 127, 128                                                # |d0| <= 127, |d1|, |d2| <= 128
    V0 = L_MAX * d0 * d0
    V1 = L_MAX * 2 * d0 * d1
    V2 = L_MAX * (2 * d0 * d1 + d1 * d1)
    T = 256 * V1 + V2
    for v in (V0, V1, V2, T):
        assert v < 2 ** 31
    assert L_MAX * (2 ** 16 * d0 * d0) + T < 2 ** 63                 # the combination itself is only ever formed in fp32
    # and one k-step more would not do for T: the bound L <= 256 is tight to within a few atoms
    assert 256 * ((L_MAX + 4) * 2 * d0 * d1) + (L_MAX + 4) * (2 * d0 * d1 + d1 * d1) >= 2 ** 31


def test_three_levels_reproduce_the_product_sum_up_to_the_dropped_levels():
    rng = np.random.default_rng(7)
    Imax = int(np.floor(KAPPA * 2 ** 23 + 0.5))
    for L in (1, 31, 100, 250, 256):
        A = rng.integers(-Imax, Imax + 1, size=(64, L))
        B = rng.integers(-Imax, Imax + 1, size=(64, L))
        a0, a1, a2 = split(A)
        b0, b1, b2 = split(B)
        exact = [sum(int(x) * int(y) for x, y in zip(ra, rb)) for ra, rb in zip(A, B)]      # Python integers: no overflow
        V0 = (a0 * b0).sum(axis=1)
        V1 = (a0 * b1 + a1 * b0).sum(axis=1)
        V2 = (a0 * b2 + a1 * b1 + a2 * b0).sum(axis=1)
        for v in (V0, V1, V2, 256 * V1 + V2):
            assert np.abs(v).max() < 2 ** 31
        kept = [(int(v0) << 32) + (int(v1) << 24) + (int(v2) << 16) for v0, v1, v2 in zip(V0, V1, V2)]
        dropped = np.array([e - k for e, k in zip(exact, kept)], dtype=np.float64)
        assert np.abs(dropped).max() <= L * (2 * 128 * 128 * 256 + 128 * 128)           # levels 3 and 4
        # relative to the scale of one product, 2^46: below 2^-21 per atom, random in sign
        assert np.abs(dropped).max() / (L * 2.0 ** 46) < 2.0 ** -21


def test_sum_of_squares_from_the_same_integers_is_exact_in_64_bits():
    Imax = int(np.floor(KAPPA * 2 ** 23 + 0.5))
    assert 3 * L_MAX * Imax * Imax < 2 ** 63                         # R^2 numerator: sum over 3 L coordinates of I^2
