"""bench.py's roofline arithmetic, checked on the host (no GPU): the algorithmic work per pair, the issued tensor work the
geometry query implies, the 8x ratio between them DESIGN.md section 7.2 derives, and the stored-traffic lookup."""
import importlib.util
import os

import pytest

import paper_1302_4000_b200 as clusco

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


PK = {"bf16_tflops": 1600.0, "hbm_gbs": 6500.0, "sm_max_mhz": 1965.0, "source": "test"}


def test_algorithmic_and_issued_work_of_the_tensor_engine(bench):
    N, L = 10000, 250
    P = N * (N - 1) // 2
    r = bench.roofline_allpairs(clusco, "C3", N, L, clusco.ENGINE_I8TC, kern_ms=0.5, step_ms=0.55, pk=PK, int8=None)
    assert r["bound"] == "tensor" and r["peak"] == 3200.0
    assert r["achieved"] == pytest.approx(18.0 * L * P / 0.5e-3 / 1e12)            # 18 L flop per pair, nothing else counted
    assert r["frac"] == pytest.approx(r["achieved"] / 3200.0)
    # six digit products x 128/96 row padding = 8, plus the diagonal tiles' and the k padding's few per cent
    assert 8.0 <= r["issued_over_algorithmic"] <= 8.0 * 1.05
    geo = clusco.i8tc_geometry(N, L)
    assert geo["ksteps"] == 8 and geo["mma_columns_per_kstep"] == 288 and (geo["row_models"], geo["col_models"]) == (32, 16)
    assert r["issued_tops"] == pytest.approx(2.0 * geo["tiles"] * 8 * 288 * 128 * 32 / 0.5e-3 / 1e12)
    assert r["algorithmic_bytes"] == 4.0 * P + 12.0 * N * L
    assert r["kernel_share_of_step"] == pytest.approx(0.5 / 0.55)


def test_cuda_core_engine_roofline_is_the_fp32_fma_peak(bench):
    r = bench.roofline_allpairs(clusco, "C3", 1000, 300, clusco.ENGINE_FFMA, kern_ms=1.0, step_ms=1.1, pk=PK, int8=None)
    assert r["bound"] == "alu" and r["peak"] == pytest.approx(148 * 128 * 2 * 1.965e9 / 1e12)


def test_stored_traffic_lookup_names_its_capture(bench):
    tr, src = bench._stored_traffic("gram_i8tc_kernel", "C3")
    assert tr is not None and tr > 0 and src.endswith("_raw.csv") and os.path.exists(os.path.join(ROOT, "profiles", src))
    assert bench._stored_traffic("no_such_kernel", "C3") == (None, None)
    assert bench.launches_per_step(clusco.ENGINE_I8TC) == 2 and bench.launches_per_step(clusco.ENGINE_FFMA) == 3
