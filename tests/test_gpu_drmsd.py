"""GPU parity of the dRMSD path (eq. 5) against the FP64 oracle (oracle/drmsd_oracle.c).

Tolerance: the paper/BASELINE state none for dRMSD; the kernel uses the same exact 24-bit fixed-point arithmetic as
the cRMSD path, so the same bar is asked: every pair |d^2_gpu - d^2_oracle| <= 2e-3 A^2 and
|d_gpu - d_oracle| <= 1e-3 A wherever d_oracle >= 0.5 A.
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


def _check(d_gpu, d_ref, d2_ref, what):
    d_gpu = np.asarray(d_gpu, np.float64)
    assert d_gpu.shape == d_ref.shape and np.all(np.isfinite(d_gpu)), what
    e2 = np.abs(d_gpu * d_gpu - d2_ref)
    assert e2.max() <= 2e-3, f"{what}: max |dd2| {e2.max():.3e}"
    big = d_ref >= 0.5
    if big.any():
        assert np.abs(d_gpu - d_ref)[big].max() <= 1e-3, what


@pytest.mark.parametrize("cfg,N", [("C1", None), ("C2", 300), ("C3", 200)])
def test_drmsd_every_pair(clusco, cfg, N):
    ens = wl.make_config(cfg, N=N)
    d_ref, d2_ref = oracle.drmsd_allpairs(ens.coords)
    got = clusco.clusco_drmsd_allpairs(_dev(ens.coords)).cpu().numpy()
    _check(got, d_ref, d2_ref, cfg)


def test_drmsd_mirrors_and_rigid_copies(clusco, c1):
    """dRMSD loses chirality: C1's mirrored decoys are as close to the rest as unmirrored ones are,
    and the two exact rigid copies of the native are at ~0."""
    got = clusco.clusco_drmsd_allpairs(_dev(c1.coords)).cpu().numpy()
    a, b = sorted(int(v) for v in c1.rigid_copy_idx[:2])
    assert got[wl.packed_index(a, b, c1.N)] < 0.05
    m = int(c1.mirror_idx[0])
    i, j = min(m, a), max(m, a)
    c = clusco.clusco_crmsd_allpairs(_dev(c1.coords)).cpu().numpy()
    assert got[wl.packed_index(i, j, c1.N)] < 0.8 * c[wl.packed_index(i, j, c1.N)]


@pytest.mark.parametrize("N,L", [(2, 2), (3, 5), (129, 33), (257, 64), (130, 296)])
def test_drmsd_ragged_shapes(clusco, N, L):
    rng = np.random.default_rng(N * 1000 + L)
    x = (rng.normal(size=(N, L, 3)) * 9 + rng.uniform(-40, 40, size=(N, 1, 3))).astype(np.float32)
    x[1] = x[0]                                                       # an identical pair: exactly 0
    d_ref, d2_ref = oracle.drmsd_allpairs(x)
    got = clusco.clusco_drmsd_allpairs(_dev(x)).cpu().numpy()
    _check(got, d_ref, d2_ref, f"N={N} L={L}")
    assert got[0] == 0.0


def test_drmsd_edge_cases(clusco):
    import torch
    x = _dev(wl.make_config("C1").coords)
    assert clusco.clusco_drmsd_allpairs(x[:1].contiguous()).numel() == 0
    one_atom = x[:5, :1, :].contiguous()
    assert torch.all(clusco.clusco_drmsd_allpairs(one_atom) == 0)
    with pytest.raises(clusco.CluscoError):
        clusco.clusco_drmsd_allpairs(torch.zeros(4, 297, 3, device="cuda"))
    y = x[:40].clone()
    y[7, 2, 0] = float("inf")
    got = clusco.clusco_drmsd_allpairs(y).cpu().numpy()
    bad = np.zeros(got.size, bool)
    for j in range(40):
        if j != 7:
            bad[wl.packed_index(min(7, j), max(7, j), 40)] = True
    assert np.all(np.isnan(got[bad])) and np.all(np.isfinite(got[~bad]))


def test_drmsd_full_size_sampled(clusco):
    """C3 at full size (10000 x 250: K = 31125, the configuration bench.py times): sampled pairs one by one."""
    ens = wl.make_config("C3")
    got = clusco.clusco_drmsd_allpairs(_dev(ens.coords)).cpu().numpy()
    rng = np.random.default_rng(7)
    pi = rng.integers(0, ens.N - 1, 20_000)
    pj = np.array([rng.integers(i + 1, ens.N) for i in pi])
    pi = np.concatenate([pi, [0, 0, ens.N - 2, 127, 128]])
    pj = np.concatenate([pj, [1, ens.N - 1, ens.N - 1, 128, 9999]])
    d_ref, d2_ref = oracle.drmsd_pairs(ens.coords, pi, pj)
    _check(got[wl.packed_index(pi, pj, ens.N)], d_ref, d2_ref, "C3 sampled")


def test_drmsd_tail_every_pair(clusco):
    """C3's recipe on the generator's most extended native (R_g^2 = 4289 A^2, the largest distances and sums)."""
    ens = wl.make_tail("C3", 400)
    d_ref, d2_ref = oracle.drmsd_allpairs(ens.coords)
    got = clusco.clusco_drmsd_allpairs(_dev(ens.coords)).cpu().numpy()
    _check(got, d_ref, d2_ref, ens.name)
    print(f"{ens.name}: max|dd2| = {np.abs(got.astype(np.float64) ** 2 - d2_ref).max():.2e}")


def test_drmsd_cluster_path_large_K_every_pair(clusco):
    """The 2 x 2 cluster kernel (N >= 897) with a long contraction: L = 160, K = 12 720 (398 k-steps, ragged last one)."""
    ens = wl.make_tail("C2", 900, 140)
    x = np.concatenate([ens.coords, ens.coords[:, :20]], axis=1).copy()        # L = 160: the chain plus a repeated piece
    d_ref, d2_ref = oracle.drmsd_allpairs(x)
    got = clusco.clusco_drmsd_allpairs(_dev(x)).cpu().numpy()
    _check(got, d_ref, d2_ref, "cluster path L=160")


def test_drmsd_cluster_path_max_L_sampled(clusco):
    """L = 296 is the int32 bound of the level sums (3 K 2^14 < 2^31): cluster path, sampled pairs, extended chains."""
    rng = np.random.default_rng(296)
    N, L = 1000, 296
    nat = wl.random_walk_chain(L, rng)
    y = nat[None] + rng.normal(size=(N, L, 3)) * rng.uniform(0.0, 3.0, size=(N, 1, 1))
    x = wl.rigid_transform(y, rng).astype(np.float32)
    x[1] = x[0]
    got = clusco.clusco_drmsd_allpairs(_dev(x)).cpu().numpy()
    pi = rng.integers(0, N - 1, 15_000)
    pj = np.array([rng.integers(i + 1, N) for i in pi])
    pi = np.concatenate([pi, [0, 0, N - 2, 127, 128]])
    pj = np.concatenate([pj, [1, N - 1, N - 1, 128, 999]])
    d_ref, d2_ref = oracle.drmsd_pairs(x, pi, pj)
    _check(got[wl.packed_index(pi, pj, N)], d_ref, d2_ref, "max L sampled")
    assert got[0] == 0.0


@pytest.mark.parametrize("N,L", [(1100, 30), (1024, 12), (2049, 20)])
def test_drmsd_cluster_path_every_pair(clusco, N, L):
    """N >= 897 (8 tiles per side) takes the 2 x 2 cluster kernel with multicast operands; T = 9 is odd, so the
    last cluster row / column hangs over the edge and the diagonal blocks hold one masked tile."""
    rng = np.random.default_rng(N + L)
    base = rng.normal(size=(1, L, 3)) * 7
    x = (base + rng.normal(size=(N, L, 3)) * rng.uniform(0.2, 3.0, size=(N, 1, 1))).astype(np.float32)
    d_ref, d2_ref = oracle.drmsd_allpairs(x)
    got = clusco.clusco_drmsd_allpairs(_dev(x)).cpu().numpy()
    _check(got, d_ref, d2_ref, f"cluster N={N} L={L}")


@pytest.mark.parametrize("N,L", [(2000, 150), (65, 33), (7, 2), (40, 300)])
def test_drmsd_and_cmo_one_vs_all(clusco, N, L):
    """The versus-reference forms: dRMSD within the pair tolerance, CMO bit-exact."""
    if L == 150:
        ens = wl.make_config("C5", N=N, chunk=N)
        native, x = ens.native, ens.coords
    else:
        rng = np.random.default_rng(L)
        native = wl.random_walk_chain(L, rng)
        x = np.stack([wl.rigid_transform((native + rng.normal(size=native.shape) * rng.uniform(0.3, 6.0))[None], rng)[0]
                      for _ in range(N)]).astype(np.float32)
        native = native.astype(np.float32)
    d_ref, d2_ref = oracle.drmsd_one_vs_all(native, x)
    got = clusco.clusco_drmsd_one_vs_all(_dev(native), _dev(x)).cpu().numpy()
    _check(got, d_ref, d2_ref, f"dRMSD one-vs-all N={N} L={L}")
    s_ref = oracle.cmo_one_vs_all(native, x, 8.0).astype(np.float32)
    s = clusco.clusco_cmo_one_vs_all(_dev(native), _dev(x), 8.0).cpu().numpy()
    assert np.array_equal(s, s_ref)
    # against itself / NaN model
    self_d = clusco.clusco_drmsd_one_vs_all(_dev(native), _dev(native[None])).cpu().numpy()
    assert self_d[0] == 0.0
    y = x[:3].copy()
    y[1, 0, 0] = np.nan
    assert np.isnan(clusco.clusco_drmsd_one_vs_all(_dev(native), _dev(y)).cpu().numpy()[1])
    assert np.isnan(clusco.clusco_cmo_one_vs_all(_dev(native), _dev(y), 8.0).cpu().numpy()[1])
