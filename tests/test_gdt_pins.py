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


# ---- the search control (fragments 4, N/4, N/2, N; re-selection below 3.5 A; "until the number of
# selected atoms does not change in four iterations").  Each pin below fails when the named constant is perturbed
# (checked with perturbed copies of gdt_oracle.c; the outcomes are quoted in the commit that added these pins). ----

def _three_segments(delta, L=60, seed=7):
    """Reference = a chain of three segments A | B | C.  Model: A unchanged, B scattered hundreds of A away, C
    translated by `delta` along the A -> C centroid axis; then a rigid motion of the whole model."""
    rng = np.random.default_rng(seed)
    a = _chain(L, seed)
    m = L // 3
    b = a.copy()
    b[m:2 * m] += rng.normal(size=(m, 3)) * 300.0 + 500.0
    axis = a[2 * m:].mean(0) - a[:m].mean(0)
    b[2 * m:] += delta * axis / np.linalg.norm(axis)
    return a.astype(np.float32), _rigid(b, rng).astype(np.float32), m


def test_reselection_cutoff_is_3_5_angstrom():
    """A seed inside A fits A exactly and leaves every atom of C at distance delta.  No contiguous fragment holds atoms
    of both A and C without a majority of scattered B atoms, so the joint fit of A u C is reached ONLY by re-selecting the
    atoms closer than 3.5 A.  delta = 3.2: C is re-selected, the joint fit (computed here by scipy) leaves every atom of
    A u C at 1.6 A: max C_2 = 2L/3.  delta = 3.8: C is never re-selected: max C_2 = L/3.  (A cut-off of 3.0 fails the
    first case, 4.5 the second.)"""
    for delta, want in ((3.2, [20, 40, 40, 40]), (3.8, [20, 20, 40, 40])):
        a, b, m = _three_segments(delta)
        idx = np.r_[0:m, 2 * m:3 * m]
        A, B = a[idx].astype(np.float64), b[idx].astype(np.float64)
        rot, _ = Rotation.align_vectors(A - A.mean(0), B - B.mean(0))
        res = np.linalg.norm((A - A.mean(0)) - rot.apply(B - B.mean(0)), axis=1)
        assert np.all((res > 1.0) & (res < 2.0)) and abs(res.mean() - delta / 2) < 1e-3      # the joint fit: delta/2 each
        s, c = oracle.gdt_pair(a, b)
        assert list(c) == want, (delta, c)
        assert s[0] == 100.0 * sum(want) / (4 * 60)


def _only_block_matches(L, start, length, run, seed):
    """Reference and model agree (up to a rigid motion) on atoms [start, start + length) only; every other atom of the
    model is scattered hundreds of A away, so a fragment that holds one of them fits nothing.  Inside the block the atoms
    come in runs of `run` coincident positions: every window SHORTER than the block then holds at most two distinct
    points (collinear: the fit's roll angle is undetermined), the whole block holds >= 3 non-collinear ones."""
    rng = np.random.default_rng(seed)
    a = _chain(L, 100 + seed) * 3.0
    pts = rng.normal(size=((length + run - 1) // run, 3)) * 25.0
    for k in range(length):
        a[start + k] = pts[k // run]
    b = a.copy()
    outside = np.ones(L, bool)
    outside[start:start + length] = False
    b[outside] += rng.normal(size=(int(outside.sum()), 3)) * 400.0 + 900.0
    return a.astype(np.float32), _rigid(b, rng).astype(np.float32)


def test_fragment_set_and_start_range():
    """Which seed fragments exist.  In each case exactly one fragment of ONE length fits more than a collinear subset:
    the count of matched atoms equals the block length if and only if that fragment is among the seeds.
    (L, start, block length, run): the last 4-window; an L/4 window in the middle and the LAST one; L/2 windows; the
    whole chain (fragment length N).  Dropping a length from {4, L/4, L/2, L}, reading L/3 for L/4, or stopping the
    start positions one short changes at least one of these counts."""
    cases = [(40, 36, 4, 1), (64, 21, 16, 4), (64, 48, 16, 4), (16, 3, 8, 3), (16, 8, 8, 3), (8, 0, 8, 3)]
    for L, start, length, run in cases:
        for seed in range(4):
            a, b = _only_block_matches(L, start, length, run, seed)
            s, c = oracle.gdt_pair(a, b)
            assert list(c) == [length] * 4, (L, start, length, seed, c)
            assert abs(s[0] - 100.0 * length / L) < 1e-12


def test_stop_rule_four_unchanged_iterations_and_seed_count():
    """Identical structures: every superposition selects all L atoms.  A seed shorter than L sees the count change once
    (len -> L) and then stay: it stops after the FOURTH unchanged count = 5 superpositions; the length-L seed after 4.
    L = 40: fragments 4, 10, 20, 40 -> 37 + 31 + 21 + 1 = 90 seeds, 89 * 5 + 4 = 449 superpositions.  (A rule of three
    unchanged counts gives 359, of five 539; a lost fragment length or start position changes the seed count.)"""
    a = _chain(40, 1).astype(np.float32)
    s, c, trace = oracle.gdt_pair_trace(a, a)
    assert trace == (90, 449, 5) and s[0] == 100.0
    a = _chain(150, 2).astype(np.float32)                      # L = 150: 4, 37, 75, 150 -> 147 + 114 + 76 + 1 seeds
    assert oracle.gdt_pair_trace(a, a)[2] == (338, 337 * 5 + 4, 5)
    a = _chain(17, 3).astype(np.float32)                       # L = 17: 4, 4 (dropped), 8, 17 -> 14 + 10 + 1 seeds
    assert oracle.gdt_pair_trace(a, a)[2] == (25, 24 * 5 + 4, 5)


def test_iteration_cap_of_20():
    """DESIGN.md section 14's reading: at most 20 superpositions per seed.  Collinear structures displaced along their
    own line reduce the search to one dimension: the fit of a selected set is the shift by the mean displacement, and
    the next set is {i : |u_i - mean| < 3.5}.  The ladder below is built so that every shift takes in exactly one more
    atom (checked here with that recurrence), so the count keeps changing and the first seed runs into the cap."""
    u = [-0.03, -0.01, 0.01, 0.03]
    sel = list(u)
    for _ in range(26):
        mu = sum(sel) / len(sel)
        u.append(mu + 3.45)                                    # just inside the new window
        sel = [x for x in u if abs(x - mu) < 3.5]
    # replay on the finished ladder from the first 4-atom seed: during the first 20 superpositions the selected count
    # never stays unchanged four times in a row (it would a few steps later) -- only a cap stops this seed at 20
    sel, counts = u[:4], [4]
    for _ in range(20):
        mu = sum(sel) / len(sel)
        sel = [x for x in u if abs(x - mu) < 3.5]
        counts.append(len(sel))
    unchanged = [p == q for p, q in zip(counts, counts[1:])]
    assert len(unchanged) == 20 and not any(all(unchanged[k:k + 4]) for k in range(17))
    L = len(u)
    a = np.zeros((L, 3))
    a[:, 0] = 50.0 * np.arange(L)
    b = a.copy()
    b[:, 0] += np.array(u)
    rng = np.random.default_rng(5)
    _, _, trace = oracle.gdt_pair_trace(a.astype(np.float32), _rigid(b, rng).astype(np.float32))
    assert trace[2] == 20


def test_cutoff_decisions_on_squared_distances_are_the_same_decisions():
    """The oracle decides sqrt(d2) < x (x = 1, 2, 3.5, 4, 8); the CUDA kernel decides d2 < x^2 without the square root
    (gdt_ova.cuh).  A decision steers the search, so the two forms must agree on EVERY double: x^2 is exact for these
    five cut-offs, the IEEE square root is monotone, so it suffices that they agree on the doubles next to x^2 -- for
    d2 <= x^2 - 8 ulp the root is below x by more than an ulp, for d2 >= x^2 it is >= x."""
    for x in (1.0, 2.0, 3.5, 4.0, 8.0):
        x2 = np.float64(x * x)
        assert float(x2) == x * x and np.sqrt(x2) == x
        lo = hi = x2
        for _ in range(8):
            lo, hi = np.nextafter(lo, 0.0), np.nextafter(hi, np.inf)
            assert (np.sqrt(lo) < x) == (lo < x2) == True     # noqa: E712
            assert (np.sqrt(hi) < x) == (hi < x2) == False    # noqa: E712
        assert np.sqrt(lo) < np.nextafter(np.float64(x), 0.0)
