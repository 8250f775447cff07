"""The seeded generator: determinism, chain geometry, config shapes, specials (DESIGN.md input recipe)."""
import numpy as np

from paper_1302_4000_b200 import workloads as wl


def test_chain_geometry():
    rng = np.random.default_rng(0)
    x = wl.random_walk_chain(250, rng)
    d = np.linalg.norm(np.diff(x, axis=0), axis=1)
    assert np.allclose(d, wl.BOND, atol=1e-9)
    u, v = x[:-2] - x[1:-1], x[2:] - x[1:-1]
    ang = np.degrees(np.arccos(np.sum(u * v, 1) / (wl.BOND ** 2)))
    assert ang.min() >= 80 - 1e-6 and ang.max() <= 150 + 1e-6
    assert np.allclose(x[:3, 2], 0.0)


def test_rotations_are_proper():
    R = wl.random_rotations(50, np.random.default_rng(1))
    assert np.allclose(np.einsum("nij,nkj->nik", R, R), np.eye(3), atol=1e-12)
    assert np.allclose(np.linalg.det(R), 1.0)


def test_C1_shape_specials_and_determinism():
    a, b = wl.make_config("C1"), wl.make_config("C1")
    assert a.coords.dtype == np.float32 and a.coords.shape == (200, 76, 3)
    assert np.array_equal(a.coords, b.coords)
    assert len(a.mirror_idx) == 5 and len(a.rigid_copy_idx) == 2
    assert np.all(a.sigma[a.rigid_copy_idx] == 0.0)
    assert not set(a.mirror_idx) & set(a.rigid_copy_idx)
    assert np.abs(a.coords).max() < 400.0
    # rigid copies keep every bond at 3.8 A (up to fp32 rounding); noisy decoys do not
    for k in a.rigid_copy_idx:
        d = np.linalg.norm(np.diff(a.coords[k].astype(np.float64), axis=0), axis=1)
        assert np.allclose(d, wl.BOND, atol=1e-4)


def test_other_config_shapes():
    c2 = wl.make_config("C2", N=64)
    assert c2.coords.shape == (64, 120, 3)
    c3 = wl.make_config("C3", N=200)
    assert c3.coords.shape == (200, 250, 3) and set(c3.cluster_id) == set(range(20))
    c4 = wl.make_config("C4", N=32)
    assert c4.coords.shape == (32, 100, 3)


def test_C5_chunks_are_independent():
    full = wl.make_config("C5", N=250, chunk=100)
    part = wl.make_config("C5", N=250, chunk=100, chunks=range(1, 3))
    assert full.coords.shape == (250, 150, 3) and full.native.shape == (150, 3)
    assert np.array_equal(full.coords[100:], part.coords)
    assert np.array_equal(full.native, part.native)


def test_packed_index_is_row_major_triu():
    N = 7
    iu = np.triu_indices(N, 1)
    assert np.array_equal(wl.packed_index(iu[0], iu[1], N), np.arange(N * (N - 1) // 2))


def test_tail_seeds_are_the_most_extended_of_200():
    """workloads.TAIL_SEEDS names, per chain length, the seed in 0..199 with the largest R_g^2 (the
    native's R_g^2 varies ~8x over seeds and the GPU path's error scales with it)."""
    for L, seed in wl.TAIL_SEEDS.items():
        rg2 = [wl.chain_shape(wl.random_walk_chain(L, np.random.default_rng(s)))["rg2"] for s in range(200)]
        assert int(np.argmax(rg2)) == seed, (L, int(np.argmax(rg2)))
    assert abs(wl.chain_shape(wl.tail_native(250))["rg2"] - 4288.75) < 0.01
    assert wl.chain_shape(wl.random_walk_chain(250, np.random.default_rng(0)))["rg2"] < np.median(rg2) * 4


def test_chain_shape_record_and_tail_ensembles():
    x = np.array([[0.0, 0, 0], [2.0, 0, 0], [0, 4.0, 0], [2.0, 4.0, 0]])           # 2 x 4 rectangle
    st = wl.chain_shape(x)
    assert np.allclose(st["gyration_eigenvalues"], [4.0, 1.0, 0.0]) and abs(st["rg2"] - 5.0) < 1e-12
    assert st["max_abs_centred"] == 2.0
    e = wl.make_tail("C3", 40)
    assert e.coords.shape == (40, 250, 3) and abs(e.stats["rg2"] - 4288.75) < 0.01
    assert not np.array_equal(e.coords[:40], wl.make_config("C3", N=40).coords)
    e5 = wl.make_tail("C5", 30)
    assert e5.coords.shape == (30, 150, 3) and e5.native.shape == (150, 3)
    assert wl.make_config("C3", N=40).stats["rg2"] < 1000.0
