"""Pins for the GDT_TS / TM-score / MaxSub oracle (oracle/gdt_oracle.c = the paper's search): closed
forms that fix the normalisation, d0, the 3.5 A selection and the percent reading; an independent library route
(scipy's Kabsch) as a lower bound; invariances."""
import numpy as np
from scipy.spatial.transform import Rotation

import oracle
from paper_1302_4000_b200 import workloads as wl


def _chain(L, seed):
    return wl.random_walk_chain(L, np.random.default_rng(seed))


def _rigid(x, rng):
    R = wl.random_rotations(1, rng)[0]
    return x.astype(np.float64) @ R.T + rng.uniform(-50, 50, size=3)


def test_identity_and_rigid_copy():
    rng = np.random.default_rng(1)
    a = _chain(60, 1).astype(np.float32)
    s, c = oracle.gdt_pair(a, a)
    assert s[0] == 100.0 and abs(s[1] - 1) < 1e-12 and abs(s[2] - 1) < 1e-12 and list(c) == [60] * 4
    b = _rigid(a, rng).astype(np.float32)
    s, c = oracle.gdt_pair(a, b)
    assert s[0] == 100.0 and s[1] > 1 - 1e-9 and s[2] > 1 - 1e-9


def test_one_displaced_atom_closed_form():
    """149 atoms identical, one moved by 50 A: the fit of the 149 leaves d = 0 for them and d = 50 for the outlier, and no
    other superposition scores higher, so TM = (149 + 1/(1 + (50/d0)^2)) / 150 with d0 = 1.24 cbrt(135) - 1.8,
    MaxSub the same with 3.5, and every C_x = 149: GDT_TS = 100 * 149 / 150."""
    L = 150
    a = _chain(L, 2).astype(np.float32)
    b = a.copy()
    b[70] += np.array([50.0, 0, 0], np.float32)
    d = float(np.linalg.norm(b[70].astype(np.float64) - a[70].astype(np.float64)))
    d0 = 1.24 * np.cbrt(L - 15.0) - 1.8
    s, c = oracle.gdt_pair(a, b)
    assert list(c) == [149] * 4 and abs(s[0] - 100.0 * 149 / 150) < 1e-12
    assert abs(s[1] - (149 + 1 / (1 + (d / d0) ** 2)) / L) < 1e-9
    assert abs(s[2] - (149 + 1 / (1 + (d / 3.5) ** 2)) / L) < 1e-9


def test_hinge_gives_half():
    """Two rigid halves, the second moved as a block far away: a superposition can match one half exactly (the length
    L/2 fragments), never both: every max C_x = L/2, GDT_TS = 50."""
    rng = np.random.default_rng(3)
    L = 40
    a = _chain(L, 3)
    b = a.copy()
    R = Rotation.from_euler("z", 100, degrees=True).as_matrix()
    b[20:] = (a[20:] - a[20:].mean(0)) @ R.T + a[20:].mean(0) + np.array([60.0, 40.0, -30.0])
    s, c = oracle.gdt_pair(a.astype(np.float32), b.astype(np.float32))
    assert list(c) == [20] * 4 and s[0] == 50.0
    assert 0.5 <= s[1] < 0.5 + 0.5 / (1 + (8 / (1.24 * np.cbrt(25.0) - 1.8)) ** 2)
    assert 0.5 <= s[2] < 0.56


def test_lower_bound_from_library_kabsch_and_invariance():
    """The length-L fragment's first superposition is the global Kabsch fit, so every score is at least its value there
    (scipy align_vectors as the independent fit); the scores do not depend on the model's frame."""
    rng = np.random.default_rng(4)
    L = 76
    a = _chain(L, 4)
    for sigma in (0.05, 1.0, 3.0):
        b = _rigid(a + rng.normal(size=a.shape) * sigma, rng)
        a32, b32 = a.astype(np.float32), b.astype(np.float32)
        A, B = a32.astype(np.float64), b32.astype(np.float64)
        rot, _ = Rotation.align_vectors(A - A.mean(0), B - B.mean(0))
        d = np.linalg.norm((A - A.mean(0)) - rot.apply(B - B.mean(0)), axis=1)
        d0 = 1.24 * np.cbrt(L - 15.0) - 1.8
        s, c = oracle.gdt_pair(a32, b32)
        for k, cut in enumerate((1, 2, 4, 8)):
            assert c[k] >= (d < cut).sum()
        assert s[1] >= (1 / (1 + (d / d0) ** 2)).mean() - 1e-9 and s[1] <= 1.0
        assert s[2] >= (1 / (1 + (d / 3.5) ** 2)).mean() - 1e-9
        if sigma == 0.05:
            assert s[0] == 100.0
        b2 = _rigid(b32, rng).astype(np.float32)               # another frame: same scores up to fp32 storage
        s2, _ = oracle.gdt_pair(a32, b2)
        assert abs(s2[1] - s[1]) < 1e-4 and abs(s2[0] - s[0]) <= 100.0 / L + 1e-9
    out = oracle.gdt_one_vs_all(a32, np.stack([b32, a32]))
    assert np.allclose(out[0], s) and out[1][0] == 100.0


def test_allpairs_form_is_symmetric_in_the_two_structures():
    """PAPER.md:84 (all-versus-all): the packed form takes model i as the reference of pair i < j.  The search selects
    atoms by distances only, so exchanging the two structures gives the same counts and scores (up to rounding of the
    inverse rotation): check the packed result against the pair routine called BOTH ways, and its shape and order."""
    rng = np.random.default_rng(11)
    a = _chain(40, 5)
    x = np.stack([_rigid(a + rng.normal(size=a.shape) * s, rng) for s in (0.0, 0.6, 1.5, 3.0, 6.0)]).astype(np.float32)
    out = oracle.gdt_allpairs(x)
    assert out.shape == (10, 3)
    k = 0
    for i in range(5):
        for j in range(i + 1, 5):
            sij, cij = oracle.gdt_pair(x[i], x[j])
            sji, cji = oracle.gdt_pair(x[j], x[i])
            assert np.allclose(out[k], sij, atol=1e-12)
            assert abs(sij[0] - sji[0]) <= 100.0 / 40 / 4 + 1e-9 and np.allclose(sij[1:], sji[1:], atol=1e-6)
            k += 1
    assert oracle.gdt_allpairs(x[:1]).shape == (0, 3)
