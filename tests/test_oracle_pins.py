"""Pins for the FP64 oracle (oracle/crmsd_oracle.c) against what the paper and the mathematics fix.

None of these re-types the oracle's formula or re-calls its routine: they are closed forms
(tests/golden/closed_forms.txt), invariants, special cases that reduce to a library routine
(LAPACK SVD, scipy's Kabsch), brute force over rotations on tiny inputs, and a statistical law.
Pin numbers P1..P15 are those of DESIGN.md / SURVEY.md section 8(c).
"""
import os

import numpy as np
import pytest

import oracle
from paper_1302_4000_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")


def _rng(seed):
    return np.random.default_rng(seed)


def _rand_model(L, rng, scale=10.0):
    return (rng.normal(size=(L, 3)) * scale + rng.uniform(-30, 30, size=3)).astype(np.float32)


def _rigid(x, rng):
    R = wl.random_rotations(1, rng)[0]
    return x.astype(np.float64) @ R.T + rng.uniform(-50, 50, size=3)


def _gyration_eigs(x):
    a = x.astype(np.float64)
    a = a - a.mean(0)
    return np.linalg.eigvalsh(a.T @ a / len(a))  # ascending


def _read_golden():
    cases, cur = [], None
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("case"):
            _, name, L, exp = line.split()
            cur = dict(name=name, L=int(L), expected=float(exp), rows=[])
            cases.append(cur)
        else:
            cur["rows"].append([float(v) for v in line.split()])
    for c in cases:
        r = np.array(c["rows"], np.float32)
        assert r.shape == (2 * c["L"], 3), c["name"]
        c["A"], c["B"] = r[: c["L"]], r[c["L"]:]
    return cases


# ---- golden closed forms (hand-derived, cited in the fixture) ----------------------------------

@pytest.mark.parametrize("case", _read_golden(), ids=lambda c: c["name"])
def test_golden_closed_forms(case):
    for fn in (oracle.crmsd_pair, oracle.crmsd_pair_eq2, oracle.crmsd_pair_eq1):
        c = fn(case["A"], case["B"])[0]
        assert abs(c - case["expected"]) < 5e-7, (fn.__name__, c)   # coords are exact in fp32
    assert abs(oracle.crmsd_pair(case["B"], case["A"])[0] - case["expected"]) < 5e-7


# ---- P1-P3: identity, rigid copy, translation ---------------------------------------------------

def test_P1_identity():
    rng = _rng(1)
    for L in (3, 17, 76, 250):
        x = _rand_model(L, rng)
        assert oracle.crmsd_pair(x, x)[0] < 1e-6


def test_P2_rigid_copy_and_P3_translation():
    rng = _rng(2)
    for L in (4, 36, 120):
        x = _rand_model(L, rng)
        y = _rigid(x, rng).astype(np.float32)               # fp32 storage rounds ~4e-6 A
        c, c2 = oracle.crmsd_pair(x, y)
        assert c < 5e-5 and c2 < 2e-9
        t = (x.astype(np.float64) + np.array([12.5, -3.25, 40.0])).astype(np.float32)
        assert oracle.crmsd_pair(x, t)[0] < 5e-5


# ---- P4, P8: mirror images (S = -1 branch) ------------------------------------------------------

def test_P4_mirror_closed_form():
    rng = _rng(4)
    for L in (5, 40, 250):
        x = _rand_model(L, rng, scale=15.0)
        m = x.astype(np.float64) * np.array([-1.0, 1.0, 1.0])
        y = _rigid(m, rng).astype(np.float32)
        g3 = _gyration_eigs(x)[0]
        c, c2, lam, S = oracle.crmsd_pair_eq2(x, y)
        assert S == -1.0
        assert abs(c - 2.0 * np.sqrt(g3)) < 1e-4
        assert abs(oracle.crmsd_pair(x, y)[0] - 2.0 * np.sqrt(g3)) < 1e-4
        assert c > 0.1                                       # chirality is kept


def test_P8_planar_mirror_is_zero():
    rng = _rng(8)
    x = _rand_model(12, rng)
    x[:, 2] = 3.0
    m = x.copy()
    m[:, 0] *= -1.0
    assert oracle.crmsd_pair(x, m)[0] < 1e-5


# ---- P5, P6: scaling ------------------------------------------------------------------------------

def test_P5_uniform_scaling_and_P6_homogeneity():
    rng = _rng(5)
    x = _rand_model(60, rng)
    rg = np.sqrt(_gyration_eigs(x).sum())
    for s in (0.5, 1.7, 3.0):
        y = (_rigid(x, rng) * 1.0)
        y = ((y - y.mean(0)) * s + y.mean(0)).astype(np.float32)
        assert abs(oracle.crmsd_pair(x, y)[0] - abs(1 - s) * rg) < 2e-4
    a, b = _rand_model(30, rng), _rand_model(30, rng)
    c = oracle.crmsd_pair(a, b)[0]
    c4 = oracle.crmsd_pair(a * np.float32(4.0), b * np.float32(4.0))[0]     # x4 is exact in fp32
    assert abs(c4 - 4.0 * c) < 1e-9


# ---- P7: two atoms / rank one ----------------------------------------------------------------------

def test_P7_two_atoms():
    rng = _rng(7)
    for _ in range(20):
        a = _rand_model(2, rng)
        b = _rand_model(2, rng)
        da = np.linalg.norm(a[0].astype(np.float64) - a[1])
        db = np.linalg.norm(b[0].astype(np.float64) - b[1])
        assert abs(oracle.crmsd_pair(a, b)[0] - abs(da - db) / 2) < 1e-9
        s, det, _ = oracle.pair_spectrum(a, b)
        assert s[1] < 1e-9 * max(s[0], 1) and abs(det) < 1e-9


# ---- P9-P11: metric properties --------------------------------------------------------------------

def test_P9_symmetry_P10_triangle_P11_bounds(c1):
    x = c1.coords[:60]
    c, c2 = oracle.crmsd_allpairs(x)
    N = x.shape[0]
    D = np.zeros((N, N))
    iu = np.triu_indices(N, 1)
    D[iu] = c                                                # row-major packed order == triu order
    D = D + D.T
    # symmetry: swap the roles explicitly
    pi, pj = iu
    cs, _ = oracle.crmsd_pairs(x, pj, pi)
    assert np.max(np.abs(cs - c)) < 1e-10
    # triangle inequality on all triples
    # D[a,c] <= D[a,b] + D[b,c]  (the property FSSS/CALIBUR/DURANDAL exploit)
    assert np.max(D[:, None, :] - (D[:, :, None] + D[None, :, :])) < 1e-9
    # bounds (R_A - R_B)^2 <= c^2 <= R_A^2 + R_B^2
    _, r2 = oracle.center(x)
    lo = (np.sqrt(r2[pi]) - np.sqrt(r2[pj])) ** 2
    hi = r2[pi] + r2[pj]
    assert np.all(c2 >= lo - 1e-9) and np.all(c2 <= hi + 1e-9)


# ---- P12: eq. 1 == eq. 2 == SVD route (the paper's central claim) ---------------------

def test_P12_three_routes_agree(c1):
    x = c1.coords
    rng = _rng(12)
    for _ in range(300):
        i, j = rng.choice(len(x), 2, replace=False)
        c_def, c2_def = oracle.crmsd_pair(x[i], x[j])
        c_e2, c2_e2, lam, S = oracle.crmsd_pair_eq2(x[i], x[j])
        c_e1, c2_e1, R = oracle.crmsd_pair_eq1(x[i], x[j])
        assert abs(c2_def - c2_e1) < 1e-9 * max(1.0, c2_def) + 1e-9
        assert abs(c2_def - c2_e2) < 1e-6          # eq. 2 loses digits in sqrt(lambda3) (squared cond.)
        assert abs(np.linalg.det(R) - 1.0) < 1e-9 and np.allclose(R @ R.T, np.eye(3), atol=1e-9)
        assert np.all(np.diff(lam) <= 0)           # descending


def test_mirror_pairs_in_C1_take_S_minus_one(c1):
    x = c1.coords
    normal = np.setdiff1d(np.arange(c1.N), c1.mirror_idx)[:10]
    for m in c1.mirror_idx:
        for n in normal:
            s, det, _ = oracle.pair_spectrum(x[m], x[n])
            assert det < 0
            c, c2 = oracle.crmsd_pair(x[m], x[n])
            _, r2 = oracle.center(x[[m, n]])
            # the S=+1 answer would be smaller by 4*s3
            assert abs((r2.sum() - 2 * (s[0] + s[1] - s[2])) - c2) < 1e-9
    a, b = c1.rigid_copy_idx[:2]
    assert oracle.crmsd_pair(x[a], x[b])[0] < 5e-5


# ---- P13: brute force over rotations on tiny inputs ------------------------------------------------

def _quat_to_R(q):
    q = q / np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def test_P13_brute_force_rotation_search():
    from scipy.optimize import minimize
    rng = _rng(13)
    grid = rng.normal(size=(4000, 4))
    grid /= np.linalg.norm(grid, axis=1, keepdims=True)
    Rs = np.array([_quat_to_R(q) for q in grid])
    for trial in range(12):
        L = int(rng.integers(3, 7))
        a32, b32 = _rand_model(L, rng, 5.0), _rand_model(L, rng, 5.0)
        if trial % 3 == 0:                                    # make some pairs near-mirror
            b32 = (a32 * np.float32([-1, 1, 1]) + rng.normal(size=(L, 3)).astype(np.float32) * np.float32(0.3))
        a = a32.astype(np.float64) - a32.astype(np.float64).mean(0)
        b = b32.astype(np.float64) - b32.astype(np.float64).mean(0)

        def msd(q):
            return np.mean(np.sum((a - b @ _quat_to_R(q).T) ** 2, axis=1))

        vals = np.mean(np.sum((a[None] - np.einsum("rij,lj->rli", Rs, b)) ** 2, axis=2), axis=1)
        best = np.inf
        for k in np.argsort(vals)[:8]:
            r = minimize(msd, grid[k], method="Nelder-Mead",
                         options=dict(xatol=1e-10, fatol=1e-13, maxiter=4000))
            best = min(best, r.fun)
        c, c2 = oracle.crmsd_pair(a32, b32)
        assert best >= c2 - 1e-9                              # nothing beats the oracle's value
        assert abs(best - c2) < 1e-6                          # and the search reaches it


# ---- O4: independent library route (LAPACK / scipy Kabsch) -----------------------------------------

def test_O4_lapack_svd_on_all_C1_pairs(c1):
    x = c1.coords.astype(np.float64)
    a = x - x.mean(1, keepdims=True)
    r2 = (a * a).sum((1, 2)) / c1.L
    M = np.einsum("ilp,jlq->ijpq", a, a) / c1.L
    s = np.linalg.svd(M, compute_uv=False)
    S = np.where(np.linalg.det(M) < 0, -1.0, 1.0)
    c2_np = np.maximum(r2[:, None] + r2[None, :] - 2 * (s[..., 0] + s[..., 1] + S * s[..., 2]), 0)
    c, c2 = oracle.crmsd_allpairs(c1.coords)
    iu = np.triu_indices(c1.N, 1)
    assert np.max(np.abs(c2 - c2_np[iu])) < 1e-9
    assert c.shape == (c1.N * (c1.N - 1) // 2,)


def test_O4_scipy_kabsch_sample(c1):
    from scipy.spatial.transform import Rotation
    x = c1.coords.astype(np.float64)
    rng = _rng(44)
    for _ in range(100):
        i, j = rng.choice(c1.N, 2, replace=False)
        a = x[i] - x[i].mean(0)
        b = x[j] - x[j].mean(0)
        _, rssd = Rotation.align_vectors(a, b)
        assert abs(rssd / np.sqrt(c1.L) - oracle.crmsd_pair(c1.coords[i], c1.coords[j])[0]) < 1e-6


def test_one_vs_all_and_rows_match_pair_route():
    ens = wl.make_config("C5", N=300, chunk=100)
    c, c2 = oracle.crmsd_one_vs_all(ens.native, ens.coords)
    for k in (0, 7, 150, 299):
        assert abs(c[k] - oracle.crmsd_pair(ens.native, ens.coords[k])[0]) < 1e-12
    x = ens.coords[:50]
    call, _ = oracle.crmsd_allpairs(x)
    crow, _ = oracle.crmsd_rows(x, 10, 20)
    lo, hi = wl.packed_index(10, 11, 50), wl.packed_index(20, 21, 50)
    assert np.array_equal(crow, call[lo:hi])
    assert abs(call[wl.packed_index(3, 17, 50)] - oracle.crmsd_pair(x[3], x[17])[0]) < 1e-12


# ---- P14: noise law (statistical) ------------------------------------------------------------------

def test_P14_noise_law():
    rng = _rng(14)
    L, sigma, n = 76, 1.0, 400
    nat = wl.random_walk_chain(L, rng)
    y = nat[None] + rng.normal(size=(n, L, 3)) * sigma
    y = wl.rigid_transform(y, rng).astype(np.float32)
    c, c2 = oracle.crmsd_one_vs_all(nat.astype(np.float32), y)
    expect = sigma ** 2 * (3 - 6 / L)
    assert abs(c2.mean() - expect) < 0.05                     # s.e. ~ 0.008 at n=400


# ---- P15: the quartic identity the GPU's Newton polish relies on ------------------------------------

def test_P15_quartic_identity(c1):
    x = c1.coords
    rng = _rng(15)
    idx = [tuple(rng.choice(c1.N, 2, replace=False)) for _ in range(200)]
    idx += [(int(m), int(n)) for m in c1.mirror_idx for n in range(3)]
    for i, j in idx:
        if i == j:
            continue
        s, det, M = oracle.pair_spectrum(x[i], x[j])
        S = 1.0 if det >= 0 else -1.0
        E = s[0] + s[1] + S * s[2]
        c2c = (M * M).sum()
        cof = np.array([np.cross(M[1], M[2]), np.cross(M[2], M[0]), np.cross(M[0], M[1])])
        c1c = (cof * cof).sum()
        f = (E * E - c2c) ** 2 - 8 * det * E - 4 * c1c
        assert abs(f) < 1e-9 * E ** 4
        fp = 4 * E * (E * E - c2c) - 8 * det
        s3 = S * s[2]
        assert abs(fp - 8 * (s[0] + s[1]) * (s[0] + s3) * (s[1] + s3)) < 1e-9 * abs(E) ** 3


def test_consumers_match_scipy_squareform(c1):
    """pairs_below / rowstats against an independent unpacking of the packed triangle (scipy's condensed order)
    and a closed form: for an ensemble of copies of ONE rigid body every c is ~0, so below = N-1 and rowsum ~ 0."""
    from scipy.spatial.distance import squareform
    x = c1.coords[:60]
    c, _ = oracle.crmsd_allpairs(x)
    D = squareform(c)                                   # full symmetric matrix, zero diagonal
    cutoff = float(np.median(c))
    rs, bl = oracle.rowstats(x, cutoff)
    assert np.allclose(rs, D.sum(axis=1), rtol=0, atol=1e-9)
    assert np.array_equal(bl, (D < cutoff).sum(axis=1) - 1)          # minus the diagonal zero
    i, j, cc = oracle.pairs_below(x, cutoff)
    iu, ju = np.nonzero(np.triu(D < cutoff, 1))
    assert np.array_equal(i, iu) and np.array_equal(j, ju) and np.allclose(cc, D[iu, ju], rtol=0, atol=0)
    assert i.size == (c < cutoff).sum() and 0 < i.size < c.size
    # closed form: rigid copies of one structure
    rng = np.random.default_rng(5)
    base = rng.normal(size=(20, 3)) * 5
    copies = np.stack([_rigid(base, rng) for _ in range(7)]).astype(np.float32)
    rs, bl = oracle.rowstats(copies, 1e-3)
    assert np.all(bl == 6) and np.all(rs < 1e-3)
    i, j, cc = oracle.pairs_below(copies, 1e-3)
    assert i.size == 21
