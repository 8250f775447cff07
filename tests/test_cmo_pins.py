"""Pins for the CMO oracle (oracle/cmo_oracle.c = the paper's eq. 6-7): hand-countable cases, a
library route (scipy pdist + numpy boolean algebra) and the properties of the Sorensen index."""
import numpy as np
from scipy.spatial.distance import pdist

import oracle
from paper_1302_4000_b200 import workloads as wl


def test_hand_counted_chain():
    # four atoms on a line at 0, 1, 2, 4; cutoff 1.5: contacts of A = {(0,1), (1,2)} -> n(A) = 2
    a = np.array([[0, 0, 0], [1, 0, 0], [2, 0, 0], [4, 0, 0]], np.float32)
    # B: 0, 1, 3, 4: contacts {(0,1), (2,3)} -> n(B) = 2, common {(0,1)} -> S = 100 * 2 * 1 / 4 = 50
    b = np.array([[0, 0, 0], [1, 0, 0], [3, 0, 0], [4, 0, 0]], np.float32)
    s, cnt = oracle.cmo_pair(a, b, 1.5)
    assert list(cnt) == [2, 2, 1] and s == 50.0
    # strict inequality of eq. 6: a distance exactly at the cut-off is NOT a contact
    s, cnt = oracle.cmo_pair(a, b, 1.0)
    assert list(cnt) == [0, 0, 0] and s == 100.0            # two empty maps: identical (reading)
    s, cnt = oracle.cmo_pair(a, a, 2.5)
    assert list(cnt) == [4, 4, 4] and s == 100.0            # (0,1) (1,2) (0,2) (2,3)


def test_identity_rigid_copy_mirror_and_bounds():
    ens = wl.make_config("C1")
    x = ens.coords
    rc = [int(v) for v in ens.rigid_copy_idx[:2]]
    s, cnt = oracle.cmo_pair(x[rc[0]], x[rc[1]], 8.0)
    assert s == 100.0 and cnt[0] == cnt[1] == cnt[2] > 75   # at least the 75 chain neighbours (3.8 A < 8 A)
    m = x[3].copy()
    m[:, 0] = -m[:, 0]
    assert oracle.cmo_pair(x[3], m, 8.0)[0] == 100.0        # contact maps, like distances, lose chirality
    s = oracle.cmo_allpairs(x[:30], 8.0)
    assert np.all((s >= 0) & (s <= 100))


def test_library_route_and_symmetry():
    ens = wl.make_config("C2", N=25)
    x = ens.coords
    cutoff = 7.5
    maps = np.stack([pdist(m.astype(np.float64)) < np.float32(cutoff) for m in x])     # condensed i<j order
    s = oracle.cmo_allpairs(x, cutoff)
    k = 0
    for i in range(25):
        for j in range(i + 1, 25):
            want = 200.0 * (maps[i] & maps[j]).sum() / (maps[i].sum() + maps[j].sum())
            assert abs(s[k] - want) < 1e-12
            assert oracle.cmo_pair(x[j], x[i], cutoff)[0] == s[k]
            k += 1
    p = oracle.cmo_pairs(x, cutoff, [0, 3], [1, 20])
    assert p[0] == s[0] and p[1] == s[wl.packed_index(3, 20, 25)]
    assert np.array_equal(oracle.cmo_rows(x, cutoff, 2, 4), s[wl.packed_index(2, 3, 25):wl.packed_index(4, 5, 25)])


def test_fp32_quotient_equals_the_rounded_fp64_quotient():
    """Host logic behind the kernel's fp32 epilogue (drmsd_i8tc.cuh): eq. 7's 200 n / (n_A + n_B) with integer counts
    (n <= K < 2^16 at L <= 296) -- the IEEE fp32 quotient of the exactly representable 200 n and n_A + n_B is the same
    float as the oracle's FP64 quotient rounded to fp32 (no double-rounding case exists for such ratios)."""
    rng = np.random.default_rng(0)
    K = 296 * 295 // 2
    den = rng.integers(1, 2 * K + 1, size=3_000_000)
    n = (rng.random(den.shape) * (den // 2 + 1)).astype(np.int64)
    a = (np.float32(200.0) * n.astype(np.float32)) / den.astype(np.float32)
    b = (200.0 * n.astype(np.float64) / den.astype(np.float64)).astype(np.float32)
    assert np.array_equal(a, b)
