"""GPU parity of the GDT_TS / TM-score / MaxSub path against the step-by-step FP64 oracle
(oracle/gdt_oracle.c).  The scores are maxima over a data-dependent series of superpositions; both sides work in
FP64 (different rotation routes: Horn quaternion + quartic Newton on the GPU, Jacobi SVD in the oracle), so the
series coincide and the bar is: GDT_TS equal to the oracle's (a count / (4 L) in fp32), TM-score and MaxSub within
2e-6 (fp32 output rounding + FP64 route differences)."""
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


def _check(got, want, what):
    got = np.asarray(got, np.float64)
    assert got.shape == want.shape and np.all(np.isfinite(got)), what
    dg = np.abs(got[:, 0] - want[:, 0])
    assert dg.max() <= 1e-4, f"{what}: GDT_TS differs by {dg.max()} at model {int(dg.argmax())}"
    assert np.abs(got[:, 1] - want[:, 1]).max() <= 2e-6, what
    assert np.abs(got[:, 2] - want[:, 2]).max() <= 2e-6, what


@pytest.mark.parametrize("N,L", [(200, 150), (150, 76), (64, 33), (40, 4), (33, 7), (20, 260)])
def test_gdt_one_vs_all(clusco, N, L):
    ens = wl.make_config("C5", N=N, chunk=N) if L == 150 else None
    if ens is not None:
        native, x = ens.native, ens.coords
    else:
        rng = np.random.default_rng(L)
        native = wl.random_walk_chain(L, rng)
        sig = rng.uniform(0.3, 6.0, size=(N, 1, 1))
        x = np.stack([wl.rigid_transform((native + rng.normal(size=native.shape) * sig[k])[None], rng)[0] for k in range(N)])
        native, x = native.astype(np.float32), x.astype(np.float32)
    want = oracle.gdt_one_vs_all(native, x)
    got = clusco.clusco_gdt_one_vs_all(_dev(native), _dev(x)).cpu().numpy()
    _check(got, want, f"N={N} L={L}")
    assert want[:, 1].min() < 0.9 and want[:, 0].max() <= 100.0


def test_gdt_closed_forms_and_edges(clusco):
    import torch
    L = 150
    a = wl.random_walk_chain(L, np.random.default_rng(2)).astype(np.float32)
    b = a.copy()
    b[70] += np.array([50.0, 0, 0], np.float32)
    x = np.stack([a, b])
    got = clusco.clusco_gdt_one_vs_all(_dev(a), _dev(x)).cpu().numpy().astype(np.float64)
    d0 = 1.24 * np.cbrt(L - 15.0) - 1.8
    assert got[0, 0] == 100.0 and abs(got[0, 1] - 1) < 1e-6 and abs(got[0, 2] - 1) < 1e-6
    assert abs(got[1, 0] - 100.0 * 149 / 150) < 1e-4
    assert abs(got[1, 1] - (149 + 1 / (1 + (50 / d0) ** 2)) / L) < 2e-6
    assert clusco.clusco_gdt_one_vs_all(_dev(a), _dev(x[:0])).shape == (0, 3)
    with pytest.raises(clusco.CluscoError):
        clusco.clusco_gdt_one_vs_all(_dev(a[:2]), _dev(x[:, :2]))
    y = x.copy()
    y[1, 3, 1] = np.nan
    got = clusco.clusco_gdt_one_vs_all(_dev(a), _dev(y)).cpu().numpy()
    assert np.all(np.isnan(got[1])) and np.all(np.isfinite(got[0]))


def test_gdt_c5_sample(clusco):
    """A 1500-model slice of C5 (the one-vs-all workload, L = 150) against the oracle, model by model."""
    ens = wl.make_config("C5", N=1500, chunk=1500)
    want = oracle.gdt_one_vs_all(ens.native, ens.coords)
    got = clusco.clusco_gdt_one_vs_all(_dev(ens.native), _dev(ens.coords)).cpu().numpy()
    _check(got, want, "C5[:1500]")


@pytest.mark.parametrize("cfg,N", [("C1", 60), ("C2", 40)])
def test_gdt_allpairs(clusco, cfg, N):
    """All-versus-all form: every pair against the oracle run pair by pair (model i as the reference)."""
    ens = wl.make_config(cfg, N=N)
    want = oracle.gdt_allpairs(ens.coords)
    got = clusco.clusco_gdt_allpairs(_dev(ens.coords)).cpu().numpy()
    _check(got, want, f"{cfg} all pairs")
    assert clusco.clusco_gdt_allpairs(_dev(ens.coords[:1])).shape == (0, 3)


def test_gdt_search_control_fixtures(clusco):
    """The fixtures that pin the oracle's search control (tests/test_gdt_pins.py), through the kernel: the 3.5 A
    re-selection cases have closed-form counts (GDT_TS = 100 * (20+40+40+40)/240 and 100 * (20+20+40+40)/240), and
    the one-displaced-atom / hinge cases of the pins are covered above."""
    from test_gdt_pins import _three_segments
    for delta, counts in ((3.2, (20, 40, 40, 40)), (3.8, (20, 20, 40, 40))):
        a, b, _ = _three_segments(delta)
        want = oracle.gdt_one_vs_all(a, b[None])
        got = clusco.clusco_gdt_one_vs_all(_dev(a), _dev(b[None])).cpu().numpy()
        _check(got, want, f"three segments, delta {delta}")
        assert abs(got[0, 0] - 100.0 * sum(counts) / 240.0) < 1e-4
