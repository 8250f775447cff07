"""GPU parity of the CMO path (eq. 6-7) against the oracle (oracle/cmo_oracle.c).

Integer work: the contact decisions are taken in FP64 with the same IEEE operations on both sides and the counts are
exact, and S = (float)(200.0 * n_AB / (n_A + n_B)) is one correctly rounded division -- so the bar is BIT-EXACT
equality with the oracle's value rounded to fp32.
"""
import numpy as np
import pytest

import oracle
from paper_1302_4000_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def clusco():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests need the B200 box")
    import paper_1302_4000_b200 as pkg
    pkg.load()
    return pkg


def _dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("cfg,N,cutoff", [("C1", None, 8.0), ("C2", 300, 6.5), ("C3", 200, 10.0), ("C1", 150, 3.9)])
def test_cmo_every_pair_bit_exact(clusco, cfg, N, cutoff):
    ens = wl.make_config(cfg, N=N)
    want = oracle.cmo_allpairs(ens.coords, cutoff).astype(np.float32)
    got = clusco.clusco_cmo_allpairs(_dev(ens.coords), cutoff).cpu().numpy()
    assert np.array_equal(got, want), (cfg, np.abs(got - want).max())
    assert want.min() < 99.0 and want.max() <= 100.0


@pytest.mark.parametrize("N,L", [(2, 2), (3, 5), (129, 33), (257, 64), (130, 296)])
def test_cmo_ragged_shapes(clusco, N, L):
    rng = np.random.default_rng(N * 1000 + L)
    x = (rng.normal(size=(N, L, 3)) * 6 + rng.uniform(-40, 40, size=(N, 1, 3))).astype(np.float32)
    x[1] = x[0]
    want = oracle.cmo_allpairs(x, 7.0).astype(np.float32)
    got = clusco.clusco_cmo_allpairs(_dev(x), 7.0).cpu().numpy()
    assert np.array_equal(got, want)
    assert got[0] == 100.0


def test_cmo_edge_cases(clusco):
    import torch
    x = _dev(wl.make_config("C1").coords)
    assert clusco.clusco_cmo_allpairs(x[:1].contiguous(), 8.0).numel() == 0
    assert torch.all(clusco.clusco_cmo_allpairs(x[:5, :1, :].contiguous(), 8.0) == 100.0)      # no atom pair
    assert torch.all(clusco.clusco_cmo_allpairs(x[:9].contiguous(), 0.0) == 100.0)             # no contact at all
    assert torch.all(clusco.clusco_cmo_allpairs(x[:9].contiguous(), 1e9) == 100.0)             # every pair in contact
    with pytest.raises(clusco.CluscoError):
        clusco.clusco_cmo_allpairs(x[:4].contiguous(), -1.0)
    y = x[:40].clone()
    y[7, 2, 0] = float("nan")
    got = clusco.clusco_cmo_allpairs(y, 8.0).cpu().numpy()
    bad = np.zeros(got.size, bool)
    for j in range(40):
        if j != 7:
            bad[wl.packed_index(min(7, j), max(7, j), 40)] = True
    assert np.all(np.isnan(got[bad])) and np.all(np.isfinite(got[~bad]))


def test_cmo_full_size_sampled(clusco):
    """C3 at full size (10000 x 250), sampled pairs one by one."""
    ens = wl.make_config("C3")
    got = clusco.clusco_cmo_allpairs(_dev(ens.coords), 8.0).cpu().numpy()
    rng = np.random.default_rng(11)
    pi = rng.integers(0, ens.N - 1, 20_000)
    pj = np.array([rng.integers(i + 1, ens.N) for i in pi])
    pi = np.concatenate([pi, [0, 0, ens.N - 2, 127, 128]])
    pj = np.concatenate([pj, [1, ens.N - 1, ens.N - 1, 128, 9999]])
    want = oracle.cmo_pairs(ens.coords, 8.0, pi, pj).astype(np.float32)
    assert np.array_equal(got[wl.packed_index(pi, pj, ens.N)], want)


def test_cmo_cluster_path_large_K_every_pair(clusco):
    """The cluster kernel (N >= 897) with a long contraction: L = 160, K = 12 720 contact bits per model."""
    ens = wl.make_tail("C2", 900, 140)
    x = np.concatenate([ens.coords, ens.coords[:, :20]], axis=1).copy()
    want = oracle.cmo_allpairs(x, 8.0).astype(np.float32)
    got = clusco.clusco_cmo_allpairs(_dev(x), 8.0).cpu().numpy()
    assert np.array_equal(got, want)


def test_cmo_cluster_path_max_L_sampled(clusco):
    """L = 296 (K = 43 660, the largest supported), cluster path, sampled pairs."""
    rng = np.random.default_rng(297)
    N, L = 1000, 296
    nat = wl.random_walk_chain(L, rng)
    y = nat[None] + rng.normal(size=(N, L, 3)) * rng.uniform(0.0, 3.0, size=(N, 1, 1))
    x = wl.rigid_transform(y, rng).astype(np.float32)
    got = clusco.clusco_cmo_allpairs(_dev(x), 8.0).cpu().numpy()
    pi = rng.integers(0, N - 1, 15_000)
    pj = np.array([rng.integers(i + 1, N) for i in pi])
    want = oracle.cmo_pairs(x, 8.0, pi, pj).astype(np.float32)
    assert np.array_equal(got[wl.packed_index(pi, pj, N)], want)


@pytest.mark.parametrize("N,L", [(1100, 30), (1024, 12), (2049, 20)])
def test_cmo_cluster_path_every_pair(clusco, N, L):
    """N >= 897 takes the 2 x 2 cluster kernel with multicast operands (odd tile count: overhanging blocks)."""
    rng = np.random.default_rng(N + L)
    base = rng.normal(size=(1, L, 3)) * 7
    x = (base + rng.normal(size=(N, L, 3)) * rng.uniform(0.2, 3.0, size=(N, 1, 1))).astype(np.float32)
    want = oracle.cmo_allpairs(x, 9.0).astype(np.float32)
    got = clusco.clusco_cmo_allpairs(_dev(x), 9.0).cpu().numpy()
    assert np.array_equal(got, want)
    assert want.min() < 90.0


@pytest.mark.parametrize("scale,shift", [(1.0, 0.0), (1.0, 4096.0), (0.1, 0.0), (0.7, -333.0)])
def test_cmo_distances_at_the_cutoff(clusco, scale, shift):
    """The prepare kernel screens eq. 6 in fp32 and falls back to the FP64 evaluation inside a narrow band around the
    cut-off: integer-lattice models have many pairs EXACTLY at the cut-off distance (3-4-0, 5-0-0, ...: strict
    inequality -> no contact) and, scaled by a non-dyadic factor, many within a few ulp of it."""
    rng = np.random.default_rng(17)
    N, L = 150, 60
    x = (rng.integers(0, 9, size=(N, L, 3)).astype(np.float64) * scale + shift).astype(np.float32)
    cutoff = float(np.float32(5.0 * scale))
    want = oracle.cmo_allpairs(x, cutoff).astype(np.float32)
    got = clusco.clusco_cmo_allpairs(_dev(x), cutoff).cpu().numpy()
    assert np.array_equal(got, want), np.abs(got - want).max()
    ova_want = oracle.cmo_one_vs_all(x[0], x[1:], cutoff).astype(np.float32)
    ova_got = clusco.clusco_cmo_one_vs_all(_dev(x[0]), _dev(x[1:]), cutoff).cpu().numpy()
    assert np.array_equal(ova_got, ova_want)
