"""Pins for the FP64 dRMSD oracle (oracle/drmsd_oracle.c = the paper's eq. 5) against what the paper
and the mathematics fix: closed forms, the chirality remark, a library route (scipy pdist) and metric properties."""
import numpy as np
import pytest
from scipy.spatial.distance import pdist

import oracle
from paper_1302_4000_b200 import workloads as wl


def _rng(seed):
    return np.random.default_rng(seed)


def _model(L, rng, scale=10.0):
    return (rng.normal(size=(L, 3)) * scale + rng.uniform(-30, 30, size=3)).astype(np.float32)


def _rigid(x, rng):
    R = wl.random_rotations(1, rng)[0]
    return x.astype(np.float64) @ R.T + rng.uniform(-50, 50, size=3)


def test_identity_and_rigid_copy():
    rng = _rng(1)
    a = _model(40, rng)
    assert oracle.drmsd_pair(a, a)[0] == 0.0
    b = _rigid(a, rng).astype(np.float32)                 # distances are invariant; fp32 storage leaves ~1e-6
    assert oracle.drmsd_pair(a, b)[0] < 2e-5


def test_mirror_image_is_zero_unlike_crmsd():
    """'dRMSD ... loses chirality': the mirror image has the same distance matrix."""
    rng = _rng(2)
    a = _model(30, rng)
    m = a.copy()
    m[:, 0] = -m[:, 0]
    assert oracle.drmsd_pair(a, m)[0] == 0.0
    assert oracle.crmsd_pair(a, m)[0] > 1.0                # cRMSD keeps chirality


def test_two_atoms_closed_form():
    a = np.array([[0, 0, 0], [3, 4, 0]], np.float32)       # d = 5
    b = np.array([[1, 1, 1], [1, 1, 3]], np.float32)       # d = 2
    d, d2 = oracle.drmsd_pair(a, b)
    assert abs(d - 3.0) < 1e-12 and abs(d2 - 9.0) < 1e-12   # K = 1: |dA - dB|
    assert oracle.drmsd_pair(a[:1], b[:1]) == (0.0, 0.0)   # a single atom has no pair


def test_uniform_scaling_closed_form():
    """B = s A: d_ij^B = s d_ij^A, and sum_{i<j} d_ij^2 = L sum_i |a_i|^2 (textbook identity), so
    dRMSD = |1 - s| R_g sqrt(2 L / (L - 1))."""
    rng = _rng(3)
    L = 25
    a = _model(L, rng)
    s = 1.375                                               # exactly representable: s*a is exact enough in fp32
    b = (a.astype(np.float64) * s).astype(np.float32)
    ad = a.astype(np.float64)
    rg2 = ((ad - ad.mean(0)) ** 2).sum() / L
    want = abs(1 - s) * np.sqrt(rg2 * 2 * L / (L - 1))
    assert abs(oracle.drmsd_pair(a, b)[0] - want) < 1e-5


def test_scipy_pdist_route_and_packed_rows():
    ens = wl.make_config("C1")
    x = ens.coords[:40]
    d, d2 = oracle.drmsd_allpairs(x)
    N, L = x.shape[0], x.shape[1]
    K = L * (L - 1) // 2
    D = np.stack([pdist(m.astype(np.float64)) for m in x])              # library distances, condensed order
    k = 0
    for i in range(N):
        for j in range(i + 1, N):
            want = np.sqrt(((D[i] - D[j]) ** 2).sum() / K)
            assert abs(d[k] - want) < 1e-9 and abs(d2[k] - want * want) < 1e-8
            k += 1
    assert k == d.size
    # rows / listed pairs agree with the whole matrix
    r, _ = oracle.drmsd_rows(x, 3, 7)
    lo = 3 * (2 * N - 3 - 1) // 2
    assert np.array_equal(r, d[lo:lo + r.size])
    p, _ = oracle.drmsd_pairs(x, [0, 5], [1, 9])
    assert p[0] == d[0] and p[1] == d[wl.packed_index(5, 9, N)]


def test_symmetry_and_triangle_inequality():
    rng = _rng(4)
    ms = [_model(20, rng) for _ in range(6)]
    for a in ms:
        for b in ms:
            dab = oracle.drmsd_pair(a, b)[0]
            assert dab == oracle.drmsd_pair(b, a)[0]
            for c in ms:
                assert dab <= oracle.drmsd_pair(a, c)[0] + oracle.drmsd_pair(c, b)[0] + 1e-12


def test_mirror_decoys_of_C1_are_close_in_drmsd_only():
    """C1's five mirror decoys (x -> -x of native + noise): dRMSD to an unmirrored decoy is small (noise only),
    cRMSD is large (S = -1 branch)."""
    ens = wl.make_config("C1")
    mi = int(ens.mirror_idx[0])
    other = int(ens.rigid_copy_idx[0])                          # an exact rigid copy of the native
    d = oracle.drmsd_pair(ens.coords[mi], ens.coords[other])[0]
    c = oracle.crmsd_pair(ens.coords[mi], ens.coords[other])[0]
    assert d < c and c > 10.0


def test_one_vs_all_forms_match_pair_route():
    ens = wl.make_config("C5", N=50, chunk=50)
    d, d2 = oracle.drmsd_one_vs_all(ens.native, ens.coords)
    s = oracle.cmo_one_vs_all(ens.native, ens.coords, 8.0)
    for n in (0, 7, 49):
        assert (d[n], d2[n]) == oracle.drmsd_pair(ens.native, ens.coords[n])
        assert s[n] == oracle.cmo_pair(ens.native, ens.coords[n], 8.0)[0]
    # closed form: the reference against itself and against its mirror image
    m = ens.native.copy()
    m[:, 2] = -m[:, 2]
    d, _ = oracle.drmsd_one_vs_all(ens.native, np.stack([ens.native, m]))
    assert d[0] == 0.0 and d[1] == 0.0
    assert list(oracle.cmo_one_vs_all(ens.native, np.stack([ens.native, m]), 8.0)) == [100.0, 100.0]
