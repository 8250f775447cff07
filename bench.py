#!/usr/bin/env python
"""bench.py -- all-vs-all cRMSD throughput on BASELINE.json's headline config (C3: N=10000, L=250), with every other
config of BASELINE.json as a side leg of the same JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload C3] [--engine auto]

A step = one pass of the whole hot path (centring + R^2, covariance/Gram, eq. 2 closed form, packed store) over one
synthetic decoy ensemble already resident in HBM.  Prints ONE JSON line (rank 0).
N > 1 (torchrun): the ranks share ONE ensemble and each computes its contiguous slice of the packed triangle
(clusco_partition_rows + clusco_crmsd_allpairs_ex); no collective on the data path; "scaling": "strong".
`--impl reference` times the FP64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "all-vs-all cRMSD pairs/sec"
UNIT = "pairs/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch, from the `ncu --set full` captures committed under profiles/
# (a STORED lookup: bench.py does not run under a profiler; the capture each figure comes from is named beside it)
STORED_TRAFFIC = os.path.join(ROOT, "profiles", "dram_traffic.csv")


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"],
                    bf16_tflops_sustained=d.get("bf16_tflops_sustained"), sm_max_mhz=d.get("sm_max_mhz", 1965.0),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=None, sm_max_mhz=1965.0,
                source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled while a region runs (B200_PROFILING.md)."""

    def __init__(self, index: int, period_ms: int = 20):
        self.rows, self.proc, self.index, self.period = [], None, index, period_ms

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", str(self.period)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            time.sleep(0.3)                       # let the first samples arrive before the region starts
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.1)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, pw, mx, reasons = [], [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_mhz_min": sm[0] if sm else None, "sm_max_mhz": mx,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


# ---- the FP64 oracle as the reported CPU baseline ---------------------------------------------------------------------

def oracle_sample(ens, seconds: float = 15.0, threads: int | None = None):
    """Time the FP64 oracle, as it stands, on the first R rows of the ensemble (about `seconds` of CPU)."""
    import oracle
    all_threads = oracle.num_threads()
    if threads is not None:
        oracle.set_num_threads(threads)
    try:
        N = ens.N
        t0 = time.perf_counter()
        c, _ = oracle.crmsd_rows(ens.coords, 0, 2)
        dt = time.perf_counter() - t0
        rate = c.size / max(dt, 1e-6)                      # includes centring all N models once
        t0 = time.perf_counter()
        c, _ = oracle.crmsd_rows(ens.coords, 0, 8)
        dt = time.perf_counter() - t0
        rate = max(rate, c.size / max(dt, 1e-6))
        rows = int(min(N - 1, max(8, seconds * rate / N)))
        t0 = time.perf_counter()
        c, _ = oracle.crmsd_rows(ens.coords, 0, rows)
        dt = time.perf_counter() - t0
        if dt < 0.6 * seconds and rows < N - 1:             # the small probes under-estimate the threaded rate: one re-run
            rows = int(min(N - 1, rows * seconds / max(dt, 1e-3)))
            t0 = time.perf_counter()
            c, _ = oracle.crmsd_rows(ens.coords, 0, rows)
            dt = time.perf_counter() - t0
        cores = oracle.num_threads()
    finally:
        oracle.set_num_threads(all_threads)
    return dict(value=c.size / dt, unit=UNIT, cores=cores, kind="oracle",
                sample=f"rows 0..{rows - 1} of {ens.name} ({c.size} pairs, {dt:.1f} s wall; FP64 Jacobi-SVD per pair, "
                       f"OpenMP over rows; centring of all {N} models included)"), c.size, dt


def run_reference(args, rank, world):
    if rank != 0:
        return
    from paper_1302_4000_b200 import workloads as wl
    ens = wl.make_config(args.workload)
    per_step_s = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(ens, per_step_s)
    tot_pairs, tot_t, last = 0, 0.0, None
    for _ in range(args.steps):
        last, n, dt = oracle_sample(ens, per_step_s)
        tot_pairs += n
        tot_t += dt
    value = tot_pairs / tot_t
    last["value"] = value
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_name(args.workload, ens), "sample": last["sample"]},
        "cpu_baseline": last,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def _workload_name(name, ens):
    P = ens.N * (ens.N - 1) // 2
    return f"{name}: N={ens.N} models x L={ens.L} C-alpha, all-vs-all packed upper triangle ({P} pairs)"


# ---- timing helpers ------------------------------------------------------------------------------------------------

def _time_calls(torch, call, reps, flush, stream, mid=False):
    """CUDA events on the launching stream around `call`, L2 flushed (untimed) before each; returns the per-call times
    (and, with mid=True, the time from the event `call` records between its two stages to the end)."""
    ev = [tuple(torch.cuda.Event(enable_timing=True) for _ in range(3)) for _ in range(reps)]
    torch.cuda.synchronize()
    for a, m, b in ev:
        if flush is not None:
            flush.zero_()
        a.record(stream)
        if mid:
            call(m)
        else:
            call()
        b.record(stream)
    torch.cuda.synchronize()
    tot = [a.elapsed_time(b) for a, m, b in ev]
    kern = [m.elapsed_time(b) for a, m, b in ev] if mid else None
    return tot, kern


def measure_int8_peak(torch, seconds=3.0):
    """Dense int8 tensor-core throughput of this GPU by the protocol of MEASURED_PEAKS.json (an 8192^3 GEMM through the
    library: torch._int_mm -> cuBLASLt), best of 10 (burst) and back to back for `seconds` (sustained)."""
    try:
        n = 8192
        a = torch.randint(-127, 127, (n, n), dtype=torch.int8, device="cuda")
        b = torch.randint(-127, 127, (n, n), dtype=torch.int8, device="cuda").t()       # column-major B
        for _ in range(3):
            torch._int_mm(a, b)
        torch.cuda.synchronize()
        ops = 2.0 * n ** 3
        best = 1e9
        for _ in range(10):
            s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s.record()
            torch._int_mm(a, b)
            e.record()
            torch.cuda.synchronize()
            best = min(best, s.elapsed_time(e))
        reps = max(10, int(seconds * 1e3 / best))
        s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s.record()
        for _ in range(reps):
            torch._int_mm(a, b)
        e.record()
        torch.cuda.synchronize()
        sus = s.elapsed_time(e) / reps
        del a, b
        return {"burst_tops": ops / (best * 1e-3) / 1e12, "sustained_tops": ops / (sus * 1e-3) / 1e12,
                "how": f"torch._int_mm int8 8192^3 (2 N^3 ops): best of 10, and {reps} back to back"}
    except Exception as ex:                                            # the library may not offer an int8 GEMM here
        return {"burst_tops": None, "sustained_tops": None, "how": f"torch._int_mm unavailable: {type(ex).__name__}: {ex}"}


def _stored_traffic(kernel, workload):
    """(bytes per launch, capture name) from profiles/dram_traffic.csv; last matching row = latest capture."""
    if not os.path.exists(STORED_TRAFFIC):
        return None, None
    best, src = None, None
    for line in open(STORED_TRAFFIC):
        f = [c.strip() for c in line.split(",")]
        if len(f) >= 4 and f[0] == kernel and f[1] == workload:
            try:
                best, src = float(f[2]) + float(f[3]), (f[4] if len(f) > 4 else "profiles/dram_traffic.csv")
            except ValueError:
                pass
    return best, src


def roofline_allpairs(clusco, name, N, L, engine, kern_ms, step_ms, pk, int8):
    """Roofline of the fused Gram + eq. 2 + store kernel.  ALGORITHMIC flops = 18 L per pair (9 L multiply-adds; upper
    triangle only -- padding rows, diagonal-tile waste and the six digit products of the exact int8 split are NOT
    counted), DESIGN.md section 7."""
    P = N * (N - 1) // 2
    flops = 18.0 * L * P
    achieved = flops / (kern_ms * 1e-3) / 1e12
    if engine == clusco.ENGINE_FFMA:
        peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12          # FP32 FFMA: #SM x 128 lanes x 2 x clock
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "peak_source": "148 SM x 128 FP32 lanes x 2 flop x sm_max_mhz (DESIGN.md 7.1)",
                "kernel": "gram_ffma_kernel"}
    else:
        peak = 2.0 * pk["bf16_tflops"]                                # int8 dense = 2x bf16 (the guide's nominal ratio)
        geo = clusco.i8tc_geometry(N, L)
        issued = 2.0 * geo["tiles"] * geo["ksteps"] * geo["mma_columns_per_kstep"] * 128 * 32
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "peak_source": f"int8 tensor peak = 2 x bf16 burst ({pk['bf16_tflops']:.0f} TFLOP/s, {pk['source']}), the "
                               "guide's nominal int8:bf16 ratio",
                "issued_tops": issued / (kern_ms * 1e-3) / 1e12,
                "issued_frac": issued / (kern_ms * 1e-3) / 1e12 / peak,
                "issued_over_algorithmic": issued / flops,
                "tile": f"{geo['row_models']} x {geo['col_models']} models",
                "kernel": "gram_i8tc_kernel"}
        if int8 and int8.get("burst_tops"):
            roof["peak_int8_measured"] = int8
            roof["frac_of_int8_measured_burst"] = achieved / int8["burst_tops"]
            roof["issued_frac_of_int8_measured_burst"] = roof["issued_tops"] / int8["burst_tops"]
            roof["issued_frac_of_int8_measured_sustained"] = roof["issued_tops"] / int8["sustained_tops"]
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["kernel_ms"] = kern_ms
    roof["kernel_share_of_step"] = kern_ms / step_ms
    tr, src = _stored_traffic(roof["kernel"], name)
    roof["traffic"] = tr
    roof["traffic_source"] = (f"stored lookup, not measured in this run: {src}" if tr is not None else None)
    roof["algorithmic_bytes"] = 4.0 * P + 12.0 * N * L
    roof["hbm_bound_ms"] = (4.0 * P + 12.0 * N * L) / (pk["hbm_gbs"] * 1e9) * 1e3
    # the epilogue's own bound: instructions per pair on the plain ALUs, at perfect issue
    roof["pairs_per_s_kernel"] = P / (kern_ms * 1e-3)
    return roof


def parity_allpairs(torch, wl, ens, out, full_limit=60_000_000, sampled=10_000_000):
    """max |dc^2| and max |dc| (c >= 0.5 A) of `out` (device, packed) against the FP64 oracle: every pair when the
    ensemble has at most `full_limit` pairs, else `sampled` random pairs plus whole rows.  Outside every timed region."""
    import numpy as np
    import oracle
    N = ens.N
    P = N * (N - 1) // 2
    worst2, worstc, checked = 0.0, 0.0, 0
    t0 = time.perf_counter()
    if P <= full_limit:
        got = out.cpu().numpy().astype(np.float64)
        bounds = list(range(0, N, 1000)) + [N]
        for lo, hi in zip(bounds, bounds[1:]):
            c_ref, c2_ref = oracle.crmsd_rows(ens.coords, lo, hi)
            k0, k1 = lo * (2 * N - lo - 1) // 2, hi * (2 * N - hi - 1) // 2
            g = got[k0:k1]
            if g.size:
                worst2 = max(worst2, float(np.abs(g * g - c2_ref).max()))
                big = c_ref >= 0.5
                if big.any():
                    worstc = max(worstc, float(np.abs(g - c_ref)[big].max()))
            checked += g.size
        how = "every pair"
    else:
        rng = np.random.default_rng(2026)
        pi = rng.integers(0, N, sampled)
        pj = rng.integers(0, N, sampled)
        keep = pi != pj
        pi, pj = np.minimum(pi, pj)[keep], np.maximum(pi, pj)[keep]
        for r in [0, 1, 127, 128, N // 2, N - 130, N - 2]:
            pi = np.concatenate([pi, np.full(N - 1 - r, r)])
            pj = np.concatenate([pj, np.arange(r + 1, N)])
        c_ref, c2_ref = oracle.crmsd_pairs(ens.coords, pi, pj)
        idx = torch.from_numpy(wl.packed_index(pi, pj, N)).cuda()
        g = out[idx].cpu().numpy().astype(np.float64)
        worst2 = float(np.abs(g * g - c2_ref).max())
        big = c_ref >= 0.5
        worstc = float(np.abs(g - c_ref)[big].max())
        checked = int(g.size)
        how = f"{sampled} random pairs + 7 whole rows"
    return {"max_dc2": worst2, "max_dc_ge_0.5": worstc, "pairs_checked": int(checked), "how": how,
            "bar": "|dc2| <= 2e-3 A^2 every pair, |dc| <= 1e-3 A for c >= 0.5 A", "pass": worst2 <= 2e-3 and worstc <= 1e-3,
            "oracle_seconds": time.perf_counter() - t0}


def time_allpairs(torch, clusco, ens, engine, steps, warmup, flush, row_begin=0, row_end=None, keep_out=False):
    """Device-resident timing of the whole hot path on `ens` (rows [row_begin,row_end) of the triangle)."""
    N, L = ens.N, ens.L
    row_end = N if row_end is None else row_end
    lo, hi = row_begin * (2 * N - row_begin - 1) // 2, row_end * (2 * N - row_end - 1) // 2
    coords = torch.from_numpy(ens.coords).cuda()
    out = torch.empty(hi - lo, dtype=torch.float32, device="cuda")
    ws = torch.empty(clusco.clusco_crmsd_allpairs_workspace(N, L), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def step(mid=None):
        # the whole hot path = clusco_crmsd_allpairs(_ex), issued as its two stages so that an event between them
        # isolates the dominant (fused Gram + eq. 2 + store) kernel inside the timed region
        clusco.clusco_allpairs_prepare(coords, ws, engine)
        if mid is not None:
            mid.record(stream)
        clusco.clusco_allpairs_compute(N, L, out, ws, engine, row_begin, row_end)

    for _ in range(warmup):
        step()
    tot, kern = _time_calls(torch, step, steps, flush, stream, mid=True)
    res = {"ms_per_step": sum(tot) / steps, "kernel_ms": sum(kern) / steps, "best_ms": min(tot), "step": step,
           "coords": coords, "out": out, "ws": ws}
    return res


def sustained_allpairs(torch, step, seconds, ms_guess, index):
    """>= `seconds` of back-to-back steps (no flush: the 200 MB of output per step exceed L2), clocks sampled under load."""
    n = max(20, int(seconds * 1e3 / max(ms_guess, 1e-3)))
    sampler = ClockSampler(index).start()
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    s.record()
    for _ in range(n):
        step()
    e.record()
    torch.cuda.synchronize()
    ms = s.elapsed_time(e) / n
    clocks = sampler.stop()
    return {"ms_per_step": ms, "steps": n, "seconds": ms * n * 1e-3, "clocks": clocks}


def rank_slice(clusco, N, world, rank):
    """Rows [row_begin, row_end) of the packed triangle owned by `rank` and the number of pairs in them."""
    bounds = clusco.clusco_partition_rows(N, world)
    lo, hi = bounds[rank], bounds[rank + 1]
    return bounds, lo, hi, hi * (2 * N - hi - 1) // 2 - lo * (2 * N - lo - 1) // 2


def combine_ranks(torch, dist, world, bounds, ms_per_step, kern_ms, my_pairs, device):
    """Job time = the slowest rank's; per-rank record for the line (what the 128-row rounding of the partition and the
    per-CTA tile split cost in balance).  One all_gather of three scalars -- timing plumbing, not a data-path collective."""
    g = torch.tensor([ms_per_step, kern_ms, float(my_pairs)], device=device, dtype=torch.float64)
    allr = [torch.zeros_like(g) for _ in range(world)]
    dist.all_gather(allr, g)
    allr = [[float(v) for v in r.tolist()] for r in allr]
    job_ms = max(r[0] for r in allr)
    per_rank = {"ms_per_step": [r[0] for r in allr], "kernel_ms": [r[1] for r in allr], "pairs": [int(r[2]) for r in allr],
                "rows": [[bounds[k], bounds[k + 1]] for k in range(world)],
                "slowest_over_fastest": job_ms / max(1e-9, min(r[0] for r in allr))}
    return job_ms, per_rank


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--engine", default="auto", choices=["auto", "ffma", "i8tc"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-ova", action="store_true", help="skip every side leg (other configs, one-vs-all, consumers, "
                                                          "dRMSD, CMO, GDT)")
    ap.add_argument("--no-parity", action="store_true", help="skip the oracle comparison of the timed outputs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import paper_1302_4000_b200 as clusco
    from paper_1302_4000_b200 import workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    clusco.load()
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    engine = {"auto": clusco.ENGINE_AUTO, "ffma": clusco.ENGINE_FFMA, "i8tc": clusco.ENGINE_I8TC}[args.engine]
    ens = wl.make_config(args.workload)
    N, L = ens.N, ens.L
    P = N * (N - 1) // 2
    if engine == clusco.ENGINE_AUTO:
        engine = clusco.ENGINE_I8TC if clusco.engine_supported(clusco.ENGINE_I8TC, L) else clusco.ENGINE_FFMA
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    pk = _peaks()

    # multi-GPU: the ranks share the ensemble; rank r owns rows [b[r], b[r+1]) of the packed triangle
    bounds, row_begin, row_end, my_pairs = rank_slice(clusco, N, world, rank)

    if dist:
        dist.barrier()
    sampler = ClockSampler(local_rank).start() if rank == 0 else None
    t = time_allpairs(torch, clusco, ens, engine, args.steps, args.warmup, flush, row_begin, row_end)
    if dist:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_per_step, kern_ms = t["ms_per_step"], t["kernel_ms"]
    per_rank = None
    if dist:
        ms_per_step, per_rank = combine_ranks(torch, dist, world, bounds, ms_per_step, kern_ms, my_pairs, "cuda")
    value = P / (ms_per_step * 1e-3)

    # e2e: host buffers, host<->device copies inside the timed region.  One GPU: the C-ABI host call.  N GPUs: every rank
    # moves the coordinates up and its own slice down around the device-pointer call (there is no collective).
    e2e = None
    if not args.no_e2e:
        h_in = torch.from_numpy(ens.coords).pin_memory()
        h_out = torch.empty(my_pairs, dtype=torch.float32).pin_memory()
        if world == 1:
            def e2e_call():
                clusco.clusco_crmsd_allpairs_host(h_in, h_out)
        else:
            d_in, d_out, d_ws = t["coords"], t["out"], t["ws"]

            def e2e_call():
                d_in.copy_(h_in, non_blocking=True)
                clusco.clusco_crmsd_allpairs(d_in, d_out, d_ws, engine, row_begin, row_end)
                h_out.copy_(d_out, non_blocking=True)
                torch.cuda.synchronize()
        e2e_call()
        reps = max(3, min(args.steps, 5))
        if dist:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(reps):
            e2e_call()
        dt = (time.perf_counter() - t0) / reps
        if dist:
            tt = torch.tensor([dt], device="cuda", dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        e2e = {"value": P / dt, "unit": UNIT, "h2d_bytes_per_step": int(N * L * 12) * world,
               "d2h_bytes_per_step": int(P * 4), "ms_per_step": dt * 1e3,
               "call": "clusco_crmsd_allpairs_host (C ABI, pinned host buffers)" if world == 1 else
                       "per rank: H2D coords, clusco_crmsd_allpairs_ex on its row slice, D2H slice"}
        del h_in, h_out

    if rank != 0:
        if dist:
            dist.barrier()
            dist.destroy_process_group()
        return

    side = not args.no_ova and world == 1
    int8 = measure_int8_peak(torch) if (engine == clusco.ENGINE_I8TC and side) else None
    roof = roofline_allpairs(clusco, args.workload, N, L, engine, kern_ms, ms_per_step, pk, int8)
    sustained = None
    parity = None
    if world == 1:
        sustained = sustained_allpairs(torch, t["step"], 2.5, ms_per_step, local_rank)
        sustained["pairs_per_s"] = P / (sustained["ms_per_step"] * 1e-3)
        if not args.no_parity:
            t["step"]()
            parity = parity_allpairs(torch, wl, ens, t["out"])

    configs = {}
    ova = consumers = drmsd = cmo = gdt = None
    if side:
        configs[args.workload] = {"ms_per_step": ms_per_step, "pairs_per_s": value, "roofline": roof, "parity": parity,
                                  "native_shape": ens.stats}
        consumers = consumers_side(torch, clusco, ens, t["coords"], t["ws"], flush, P, ms_per_step, args.no_e2e)
        coords_main, out_main = t["coords"], t["out"]
        del t
        # CMO before dRMSD: the dRMSD Gram holds the GPU at its power cap for ~50 ms and whatever is timed right after it
        # runs at the reduced clock
        if L <= 296:
            cmo = cmo_side(torch, clusco, coords_main, out_main, flush, N, L, P, pk)
            drmsd = drmsd_side(torch, clusco, coords_main, out_main, flush, N, L, P, pk)
        del coords_main, out_main
        torch.cuda.empty_cache()
        for name in ("C1", "C2", "C4"):
            if name == args.workload:
                continue
            configs[name] = config_side(torch, clusco, wl, name, pk, int8, flush, args.no_parity)
            torch.cuda.empty_cache()
        ova = one_vs_all_side(torch, clusco, wl, pk, flush, args.no_parity)
        configs["C5"] = ova
        gdt = gdt_side(torch, clusco, wl)

    cpu = cpu1 = None
    if not args.no_cpu_baseline:
        cpu, _, _ = oracle_sample(ens, 12.0)
        cpu1, _, _ = oracle_sample(ens, 8.0, threads=1)

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "strong" if world > 1 else "weak",
        "vs_baseline": None, "dtype": "f32" if engine == clusco.ENGINE_FFMA else "s8",
        "data": "synthetic",
        "config": {"workload": _workload_name(args.workload, ens) +
                               (f", ONE ensemble, row-partitioned over {world} GPUs (clusco_partition_rows)" if world > 1 else ""),
                   "engine": {1: "ffma", 2: "i8tc"}[engine], "l2": "flushed between timed iterations (256 MB write)",
                   "effective_tflops": 18.0 * L * P / (ms_per_step * 1e-3) / 1e12,
                   "native_shape": ens.stats},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step(engine) * args.steps,
        "roofline": roof, "parity": parity, "sustained": sustained, "per_rank": per_rank,
        "cpu_baseline": cpu, "cpu_baseline_1thread": cpu1,
        "configs": configs or None, "one_vs_all": ova, "consumers": consumers, "drmsd": drmsd, "cmo": cmo, "gdt": gdt,
    }))
    if dist:
        dist.barrier()
        dist.destroy_process_group()


def config_side(torch, clusco, wl, name, pk, int8, flush, no_parity):
    """One more config of BASELINE.json through the same path: time, roofline (algorithmic + issued), parity."""
    ens = wl.make_config(name)
    N, L = ens.N, ens.L
    P = N * (N - 1) // 2
    engine = clusco.ENGINE_I8TC if clusco.engine_supported(clusco.ENGINE_I8TC, L) else clusco.ENGINE_FFMA
    steps = 200 if P < 5_000_000 else 20                                 # >= 200 repetitions for C1-C2
    t = time_allpairs(torch, clusco, ens, engine, steps, 3, flush)
    roof = roofline_allpairs(clusco, name, N, L, engine, t["kernel_ms"], t["ms_per_step"], pk, int8)
    par = None
    if not no_parity:
        t["step"]()
        par = parity_allpairs(torch, wl, ens, t["out"])
    return {"workload": _workload_name(name, ens), "steps": steps, "ms_per_step": t["ms_per_step"], "best_ms": t["best_ms"],
            "pairs_per_s": P / (t["ms_per_step"] * 1e-3), "roofline": roof, "parity": par, "native_shape": ens.stats}


def one_vs_all_side(torch, clusco, wl, pk, flush, no_parity):
    """Step a6 on its own workload (C5: one native vs 10^6 models x 150 atoms, 1.8 GB): HBM-bound single pass."""
    import numpy as np
    N, L, chunk = 1_000_000, 150, 100_000
    ens0 = wl.make_config("C5", N=N, chunk=chunk, chunks=range(0))
    coords = torch.empty((N, L, 3), dtype=torch.float32, device="cuda")
    first = None
    for k in range(N // chunk):
        part = wl.make_config("C5", N=N, chunk=chunk, chunks=range(k, k + 1))
        coords[k * chunk:(k + 1) * chunk] = torch.from_numpy(part.coords).cuda()
        if k == 0:
            first = part.coords
    native = torch.from_numpy(ens0.native).cuda()
    out = torch.empty(N, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(3):
        clusco.clusco_crmsd_one_vs_all(native, coords, out)
    tot, _ = _time_calls(torch, lambda: clusco.clusco_crmsd_one_vs_all(native, coords, out), 10, flush, stream)
    ms = sum(tot) / len(tot)
    nbytes = 12.0 * N * L + 4.0 * N
    gbs = nbytes / (ms * 1e-3) / 1e9
    par = None
    if not no_parity:
        import oracle
        t0 = time.perf_counter()
        c_ref, c2_ref = oracle.crmsd_one_vs_all(ens0.native, first)
        g = out[:chunk].cpu().numpy().astype(np.float64)
        big = c_ref >= 0.5
        par = {"max_dc2": float(np.abs(g * g - c2_ref).max()), "max_dc_ge_0.5": float(np.abs(g - c_ref)[big].max()),
               "pairs_checked": int(chunk), "how": "models 0..99999", "oracle_seconds": time.perf_counter() - t0}
        par["pass"] = par["max_dc2"] <= 2e-3 and par["max_dc_ge_0.5"] <= 1e-3
    tr, src = _stored_traffic("one_vs_all_stream_kernel", "C5")
    # steps a1 + a2 on their own (the public clusco_center), on the same resident coordinates: read once, write once
    centred = torch.empty_like(coords)
    r2 = torch.empty(N, dtype=torch.float32, device="cuda")
    for _ in range(3):
        clusco.clusco_center(coords, centred, r2)
    ctot, _ = _time_calls(torch, lambda: clusco.clusco_center(coords, centred, r2), 10, flush, stream)
    cms = sum(ctot) / len(ctot)
    cbytes = 24.0 * N * L + 4.0 * N
    cpar = None
    if not no_parity:
        import oracle
        cen_ref, r2_ref = oracle.center(first[:20000])
        cpar = {"max_abs_centred": float(np.abs(centred[:20000].cpu().numpy().astype(np.float64) - cen_ref).max()),
                "max_rel_r2": float(np.abs(r2[:20000].cpu().numpy().astype(np.float64) / r2_ref - 1.0).max()),
                "models_checked": 20000}
        cpar["pass"] = cpar["max_abs_centred"] <= 1e-5 and cpar["max_rel_r2"] <= 1e-6
    center = {"workload": "clusco_center on the same 10^6 x 150 coordinates", "ms": cms, "models_per_s": N / (cms * 1e-3),
              "roofline": {"bound": "hbm", "achieved": cbytes / (cms * 1e-3) / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
                           "frac": cbytes / (cms * 1e-3) / 1e9 / pk["hbm_gbs"], "algorithmic_bytes": cbytes,
                           "kernel": "center_kernel"}, "parity": cpar}
    del centred
    return {"workload": "C5: 1 native vs N=1000000 models x L=150", "ms": ms, "models_per_s": N / (ms * 1e-3),
            "center": center,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / pk["hbm_gbs"], "traffic": tr,
                         "traffic_source": f"stored lookup, not measured in this run: {src}" if tr else None,
                         "algorithmic_bytes": nbytes, "kernel": "one_vs_all_stream_kernel"},
            "parity": par, "native_shape": ens0.stats}


def consumers_side(torch, clusco, ens, coords, ws, flush, P, store_ms, no_e2e):
    """NEXT-1: the same pass with the matrix consumed in the epilogue instead of stored --
    pairs below 3.2 A (the paper's cut-off) compacted, and per-model row sums / neighbour counts;
    device-resident, and end to end through the host-buffer C-ABI calls (coordinates up, triples / statistics down)."""
    stream = torch.cuda.current_stream()
    res = {}
    for name, call in (("below_3.2A", lambda: clusco.clusco_crmsd_allpairs_below(coords, 3.2, 1 << 22, workspace=ws)),
                       ("rowstats_3.2A", lambda: clusco.clusco_crmsd_rowstats(coords, 3.2, workspace=ws))):
        for _ in range(3):
            r = call()
        tot, _ = _time_calls(torch, call, 10, flush, stream)
        ms = sum(tot) / len(tot)
        res[name] = {"ms": ms, "pairs_per_s": P / (ms * 1e-3), "vs_store_step": ms / store_ms}
        if name.startswith("below"):
            res[name]["pairs_found"] = int(r[3].item())
    if not no_e2e:
        h_in = torch.from_numpy(ens.coords).pin_memory()
        cap = 1 << 22
        bufs = (torch.empty(cap, dtype=torch.int32).pin_memory(), torch.empty(cap, dtype=torch.int32).pin_memory(),
                torch.empty(cap, dtype=torch.float32).pin_memory())
        rs = (torch.empty(ens.N, dtype=torch.float64).pin_memory(), torch.empty(ens.N, dtype=torch.int32).pin_memory())
        for name, call, down in (
                ("below_3.2A", lambda: clusco.clusco_crmsd_allpairs_below_host(h_in, 3.2, cap, out=bufs), None),
                ("rowstats_3.2A", lambda: clusco.clusco_crmsd_rowstats_host(h_in, 3.2, out=rs), ens.N * 12)):
            r = call()
            t0 = time.perf_counter()
            for _ in range(5):
                r = call()
            dt = (time.perf_counter() - t0) / 5
            d2h = down if down is not None else 8 + 12 * min(cap, r[3])
            res[name]["e2e"] = {"value": P / dt, "unit": UNIT, "ms_per_step": dt * 1e3,
                                "h2d_bytes_per_step": int(ens.N * ens.L * 12), "d2h_bytes_per_step": int(d2h),
                                "call": f"clusco_crmsd_{'allpairs_below' if down is None else 'rowstats'}_host"}
    return res


def drmsd_side(torch, clusco, coords, out, flush, N, L, P, pk):
    """NEXT-2: all-vs-all dRMSD (eq. 5) on the same ensemble -- one int8 tensor-core Gram over the
    K = L(L-1)/2 distances per model.  Algorithmic work = 2 K flop per pair (one multiply-add per distance)."""
    stream = torch.cuda.current_stream()
    K = L * (L - 1) // 2
    ws = torch.empty(int(clusco.load().clusco_drmsd_allpairs_workspace(N, L)), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        clusco.clusco_drmsd_allpairs(coords, out, ws)
    tot, _ = _time_calls(torch, lambda: clusco.clusco_drmsd_allpairs(coords, out, ws), 5, flush, stream)
    ms = sum(tot) / len(tot)
    flops = 2.0 * K * P
    peak = 2.0 * pk["bf16_tflops"]
    Np = (N + 127) // 128 * 128
    T = Np // 128
    issued = 2.0 * (T * (T + 1) // 2) * ((K + 31) // 32) * 128 * (6 * 128) * 32        # 2 x N=256 + 2 x N=128 MMAs per k-step (= six N=128 products)
    return {"workload": f"dRMSD all-vs-all, N={N} x L={L} (K={K} distances per model)", "ms": ms,
            "pairs_per_s": P / (ms * 1e-3),
            "roofline": {"bound": "tensor", "achieved": flops / (ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                         "frac": flops / (ms * 1e-3) / 1e12 / peak,
                         "issued_frac": issued / (ms * 1e-3) / 1e12 / peak, "kernel": "drmsd_gram_kernel<3,2,2,1> (+ drmsd_prep_kernel<3>)",
                         "workspace_bytes": int(ws.numel())}}


def cmo_side(torch, clusco, coords, out, flush, N, L, P, pk):
    """NEXT-3: all-vs-all contact map overlap (eq. 6-7, cut-off 8 A) on the same ensemble -- a 0/1
    int8 tensor-core Gram over the K = L(L-1)/2 contact bits per model (one byte per contact bit); roofline: the int8
    tensor pipe, 2 K operations per pair."""
    stream = torch.cuda.current_stream()
    K = L * (L - 1) // 2
    ws = torch.empty(int(clusco.load().clusco_cmo_allpairs_workspace(N, L)), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        clusco.clusco_cmo_allpairs(coords, 8.0, out, ws)
    tot, _ = _time_calls(torch, lambda: clusco.clusco_cmo_allpairs(coords, 8.0, out, ws), 5, flush, stream)
    ms = sum(tot) / len(tot)
    ops = 2.0 * K * P                                   # one AND + one add per contact bit and pair
    peak = 2.0 * pk["bf16_tflops"]
    return {"workload": f"CMO all-vs-all, cut-off 8 A, N={N} x L={L} (K={K} contact bits per model)", "ms": ms,
            "pairs_per_s": P / (ms * 1e-3),
            "roofline": {"bound": "tensor", "achieved": ops / (ms * 1e-3) / 1e12, "peak": peak, "unit": "TOP/s",
                         "frac": ops / (ms * 1e-3) / 1e12 / peak, "kernel": "drmsd_gram_kernel<1,1,2,2> (+ drmsd_prep_kernel<1>)",
                         "workspace_bytes": int(ws.numel())}}


def gdt_side(torch, clusco, wl):
    """NEXT-4: GDT_TS / TM-score / MaxSub of the first 20 000 models of C5 (L=150) against the native --
    the paper's fragment-seeded iterative search, FP64, one warp per model.  Data-dependent work: reported as models/s."""
    N = 20_000
    ens = wl.make_config("C5", N=N, chunk=N)
    native = torch.from_numpy(ens.native).cuda()
    coords = torch.from_numpy(ens.coords).cuda()
    out = torch.empty((N, 3), dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    clusco.clusco_gdt_one_vs_all(native, coords, out)
    tot, _ = _time_calls(torch, lambda: clusco.clusco_gdt_one_vs_all(native, coords, out), 3, None, stream)
    ms = sum(tot) / len(tot)
    o = out.cpu().numpy()
    # all-versus-all form on the first 200 of those models: 19 900 pairs, one warp per pair
    M = 200
    sub = coords[:M].contiguous()
    ap = clusco.clusco_gdt_allpairs(sub)
    tot, _ = _time_calls(torch, lambda: clusco.clusco_gdt_allpairs(sub, ap), 1, None, stream)
    ms_ap = tot[0]
    return {"workload": f"GDT_TS / TM-score / MaxSub, 1 native vs first {N} models of C5 (L=150)", "ms": ms,
            "models_per_s": N / (ms * 1e-3), "mean_gdt_ts": float(o[:, 0].mean()), "mean_tm_score": float(o[:, 1].mean()),
            "kernel": "gdt_kernel<false>", "bound": "alu (FP64, data-dependent iteration count)",
            "allpairs": {"workload": f"all-vs-all over the first {M} of those models ({M * (M - 1) // 2} pairs)", "ms": ms_ap,
                         "pairs_per_s": M * (M - 1) // 2 / (ms_ap * 1e-3), "kernel": "gdt_kernel<true>"}}


def launches_per_step(engine):
    # i8tc: i8_prep_kernel (centring + R^2 + operand images) and gram_i8tc_kernel (Gram + eq. 2 + packed store);
    # ffma: model_stats_kernel, ffma_plane_kernel, gram_ffma_kernel
    return 2 if engine == 2 else 3


if __name__ == "__main__":
    main()
