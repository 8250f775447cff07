#!/usr/bin/env python
"""bench.py -- all-vs-all cRMSD throughput on BASELINE.json's headline config (C3: N=10000, L=250).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload C3] [--engine auto]

A step = one pass of the whole hot path (centring + R^2, covariance/Gram, eq. 2 closed form, packed
store) over one synthetic decoy ensemble already resident in HBM.  Prints ONE JSON line (rank 0).
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


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], sm_max_mhz=d.get("sm_max_mhz", 1965.0),
                    source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled during the timed region (B200_PROFILING.md)."""

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_sample(ens, seconds: float = 15.0):
    """Time the FP64 oracle, as it stands, on the first R rows of the ensemble (about `seconds` of CPU)."""
    import oracle
    N = ens.N
    t0 = time.perf_counter()
    c, _ = oracle.crmsd_rows(ens.coords, 0, 2)
    probe_rows = 2
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
    del probe_rows
    return dict(value=c.size / dt, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
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
        "config": {"workload": f"{args.workload}: N={ens.N} models x L={ens.L} C-alpha, all-vs-all",
                   "sample": last["sample"]},
        "cpu_baseline": last,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--engine", default="auto", choices=["auto", "ffma", "i8tc"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-ova", action="store_true", help="skip the one-vs-all (C5) side measurement")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import numpy as np
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
    # one independent ensemble per rank (the paper clusters 56 targets independently):
    # rank r perturbs nothing but owns its own copy of the workload -> weak scaling, no collective.
    ens = wl.make_config(args.workload)
    N, L = ens.N, ens.L
    P = N * (N - 1) // 2
    if engine == clusco.ENGINE_AUTO:
        engine = clusco.ENGINE_I8TC if clusco.engine_supported(clusco.ENGINE_I8TC, L) else clusco.ENGINE_FFMA
    coords = torch.from_numpy(ens.coords).cuda()
    out = torch.empty(P, dtype=torch.float32, device="cuda")
    ws = torch.empty(clusco.clusco_crmsd_allpairs_workspace(N, L), dtype=torch.uint8, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step(mid=None):
        # the whole hot path = clusco_crmsd_allpairs, issued as its two stages so that an event between
        # them isolates the dominant (fused Gram + eq. 2 + store) kernel inside the timed region
        clusco.clusco_allpairs_prepare(coords, ws, engine)
        if mid is not None:
            mid.record(stream)
        clusco.clusco_allpairs_compute(N, L, out, ws, engine)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev = [tuple(torch.cuda.Event(enable_timing=True) for _ in range(3)) for _ in range(args.steps)]
    torch.cuda.synchronize()
    for a, m, b in ev:
        flush.zero_()                                   # L2 flush between timed iterations (untimed)
        a.record(stream)
        step(m)
        b.record(stream)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    total_ms = sum(a.elapsed_time(b) for a, m, b in ev)
    kern_ms = sum(m.elapsed_time(b) for a, m, b in ev) / args.steps
    clocks = sampler.stop() if rank == 0 else None
    if dist:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = world * P / (ms_per_step * 1e-3)

    # e2e: the host-buffer C-ABI call, host<->device copies inside the timed region
    e2e = None
    if not args.no_e2e:
        h_in = torch.from_numpy(ens.coords).pin_memory()
        h_out = torch.empty(P, dtype=torch.float32).pin_memory()
        clusco.clusco_crmsd_allpairs_host(h_in, h_out)
        reps = max(2, min(args.steps, 5))
        if dist:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(reps):
            clusco.clusco_crmsd_allpairs_host(h_in, h_out)
        dt = (time.perf_counter() - t0) / reps
        if dist:
            t = torch.tensor([dt], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * P / dt, "unit": UNIT, "h2d_bytes_per_step": int(N * L * 12),
               "d2h_bytes_per_step": int(P * 4), "ms_per_step": dt * 1e3}

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    # roofline for the dominant kernel (the fused Gram + eq. 2 + store kernel): ALGORITHMIC flops = 18 L per pair
    # (9 L multiply-adds; upper triangle only -- padding rows, diagonal-tile waste and the six digit products of
    # the exact int8 split are NOT counted), DESIGN.md section 7
    pk = _peaks()
    flops = 18.0 * L * P
    achieved = flops / (kern_ms * 1e-3) / 1e12
    if engine == clusco.ENGINE_FFMA:
        peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12          # FP32 FFMA: #SM x 128 lanes x 2 x clock
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "peak_source": "148 SM x 128 FP32 lanes x 2 flop x sm_max_mhz (DESIGN.md 7.1)"}
    else:
        peak = 2.0 * pk["bf16_tflops"]                                # int8 dense = 2x bf16 (the guide's nominal ratio)
        # what the tensor pipe actually executes: tiles x k-steps x (144+96+48) columns x 128 rows x 32 atoms
        Tc, Tr, ks = (N + 15) // 16, (N + 31) // 32, (L + 31) // 32
        tiles = sum(Tc - 2 * i for i in range(Tr))
        issued = 2.0 * tiles * ks * 288 * 128 * 32
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "peak_source": f"int8 tensor peak = 2 x {pk['source']} bf16 burst ({pk['bf16_tflops']:.0f} TFLOP/s), "
                               "nominal int8:bf16 ratio (of measured)",
                "issued_tops": issued / (kern_ms * 1e-3) / 1e12,
                "issued_frac": issued / (kern_ms * 1e-3) / 1e12 / peak,
                "issued_over_algorithmic": issued / flops}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["kernel_ms"] = kern_ms
    roof["kernel"] = "gram_ffma_kernel" if engine == clusco.ENGINE_FFMA else "gram_i8tc_kernel"
    roof["kernel_share_of_step"] = kern_ms / ms_per_step
    roof["traffic"] = _ncu_traffic(roof["kernel"], args.workload)
    roof["algorithmic_bytes"] = 4.0 * P + 12.0 * N * L
    roof["hbm_bound_ms"] = (4.0 * P + 12.0 * N * L) / (pk["hbm_gbs"] * 1e9) * 1e3

    ova = None
    if not args.no_ova and world == 1:
        ova = one_vs_all_side(clusco, wl, pk, flush)
    consumers = None
    drmsd = None
    cmo = None
    gdt = None
    if not args.no_ova and world == 1:
        consumers = consumers_side(clusco, coords, ws, flush, P, ms_per_step)
        del ws
        # CMO before dRMSD: the dRMSD Gram holds the GPU at its power cap for ~50 ms and whatever is timed right after it
        # runs at the reduced clock (CMO read 2.05 ms after it, 1.67 ms before it or alone)
        cmo = cmo_side(clusco, coords, out, flush, N, L, P, pk)
        drmsd = drmsd_side(clusco, coords, out, flush, N, L, P, pk)
        gdt = gdt_side(clusco, wl)

    cpu = None
    if not args.no_cpu_baseline:
        cpu, _, _ = oracle_sample(ens, 15.0)

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if engine == clusco.ENGINE_FFMA else "s8",
        "data": "synthetic",
        "config": {"workload": f"{args.workload}: N={N} models x L={L} C-alpha, all-vs-all packed upper triangle "
                               f"({P} pairs), one ensemble per GPU",
                   "engine": {1: "ffma", 2: "i8tc"}[engine], "l2": "flushed between timed iterations (256 MB write)",
                   "effective_tflops": flops * world / (ms_per_step * 1e-3) / 1e12},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step(engine) * args.steps,
        "roofline": roof, "cpu_baseline": cpu, "one_vs_all": ova, "consumers": consumers, "drmsd": drmsd, "cmo": cmo, "gdt": gdt,
    }))
    if dist:
        dist.destroy_process_group()


def _ncu_traffic(kernel, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return None
    best = None
    for line in open(path):
        f = [c.strip() for c in line.split(",")]
        if len(f) >= 4 and f[0] == kernel and f[1] == workload:
            best = float(f[2]) + float(f[3])          # last matching row = latest round
    return best


def one_vs_all_side(clusco, wl, pk, flush):
    """Step a6 on its own workload (C5: one native vs 10^6 models x 150 atoms, 1.8 GB): HBM-bound single pass."""
    import torch
    N, L, chunk = 1_000_000, 150, 100_000
    ens0 = wl.make_config("C5", N=N, chunk=chunk, chunks=range(0))
    coords = torch.empty((N, L, 3), dtype=torch.float32, device="cuda")
    for k in range(N // chunk):
        part = wl.make_config("C5", N=N, chunk=chunk, chunks=range(k, k + 1))
        coords[k * chunk:(k + 1) * chunk] = torch.from_numpy(part.coords).cuda()
    native = torch.from_numpy(ens0.native).cuda()
    out = torch.empty(N, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(3):
        clusco.clusco_crmsd_one_vs_all(native, coords, out)
    reps = 10
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    torch.cuda.synchronize()
    for a, b in ev:
        flush.zero_()                                   # inputs (1.8 GB) exceed L2 anyway
        a.record(stream)
        clusco.clusco_crmsd_one_vs_all(native, coords, out)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / reps
    nbytes = 12.0 * N * L + 4.0 * N
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"workload": "C5: 1 native vs N=1000000 models x L=150", "ms": ms, "models_per_s": N / (ms * 1e-3),
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / pk["hbm_gbs"], "traffic": _ncu_traffic("one_vs_all_stream_kernel", "C5"),
                         "algorithmic_bytes": nbytes, "kernel": "one_vs_all_stream_kernel"}}


def consumers_side(clusco, coords, ws, flush, P, store_ms):
    """NEXT-1: the same pass with the matrix consumed in the epilogue instead of stored --
    pairs below 3.2 A (the paper's cut-off) compacted, and per-model row sums / neighbour counts."""
    import torch
    stream = torch.cuda.current_stream()
    res = {}
    for name, call in (("below_3.2A", lambda: clusco.clusco_crmsd_allpairs_below(coords, 3.2, 1 << 22, workspace=ws)),
                       ("rowstats_3.2A", lambda: clusco.clusco_crmsd_rowstats(coords, 3.2, workspace=ws))):
        for _ in range(3):
            r = call()
        reps = 10
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        torch.cuda.synchronize()
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            r = call()
            b.record(stream)
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev) / reps
        res[name] = {"ms": ms, "pairs_per_s": P / (ms * 1e-3), "vs_store_step": ms / store_ms}
        if name.startswith("below"):
            res[name]["pairs_found"] = int(r[3].item())
    return res


def drmsd_side(clusco, coords, out, flush, N, L, P, pk):
    """NEXT-2: all-vs-all dRMSD (eq. 5) on the same ensemble -- one int8 tensor-core Gram over the
    K = L(L-1)/2 distances per model.  Algorithmic work = 2 K flop per pair (one multiply-add per distance)."""
    import torch
    stream = torch.cuda.current_stream()
    K = L * (L - 1) // 2
    ws = torch.empty(int(clusco.load().clusco_drmsd_allpairs_workspace(N, L)), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        clusco.clusco_drmsd_allpairs(coords, out, ws)
    reps = 5
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    torch.cuda.synchronize()
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        clusco.clusco_drmsd_allpairs(coords, out, ws)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / reps
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


def cmo_side(clusco, coords, out, flush, N, L, P, pk):
    """NEXT-3: all-vs-all contact map overlap (eq. 6-7, cut-off 8 A) on the same ensemble -- a 0/1
    int8 tensor-core Gram over the K = L(L-1)/2 contact bits per model (one byte per contact bit); roofline: the int8
    tensor pipe, 2 K operations per pair."""
    import torch
    stream = torch.cuda.current_stream()
    K = L * (L - 1) // 2
    ws = torch.empty(int(clusco.load().clusco_cmo_allpairs_workspace(N, L)), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        clusco.clusco_cmo_allpairs(coords, 8.0, out, ws)
    reps = 5
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    torch.cuda.synchronize()
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        clusco.clusco_cmo_allpairs(coords, 8.0, out, ws)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / reps
    ops = 2.0 * K * P                                   # one AND + one add per contact bit and pair
    peak = 2.0 * pk["bf16_tflops"]
    return {"workload": f"CMO all-vs-all, cut-off 8 A, N={N} x L={L} (K={K} contact bits per model)", "ms": ms,
            "pairs_per_s": P / (ms * 1e-3),
            "roofline": {"bound": "tensor", "achieved": ops / (ms * 1e-3) / 1e12, "peak": peak, "unit": "TOP/s",
                         "frac": ops / (ms * 1e-3) / 1e12 / peak, "kernel": "drmsd_gram_kernel<1,1,2,2> (+ drmsd_prep_kernel<1>)",
                         "workspace_bytes": int(ws.numel())}}


def gdt_side(clusco, wl):
    """NEXT-4: GDT_TS / TM-score / MaxSub of the first 20 000 models of C5 (L=150) against the native --
    the paper's fragment-seeded iterative search, FP64, one warp per model.  Data-dependent work: reported as models/s."""
    import torch
    N = 20_000
    ens = wl.make_config("C5", N=N, chunk=N)
    native = torch.from_numpy(ens.native).cuda()
    coords = torch.from_numpy(ens.coords).cuda()
    out = torch.empty((N, 3), dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    clusco.clusco_gdt_one_vs_all(native, coords, out)
    reps = 3
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    torch.cuda.synchronize()
    for a, b in ev:
        a.record(stream)
        clusco.clusco_gdt_one_vs_all(native, coords, out)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / reps
    o = out.cpu().numpy()
    # all-versus-all form on the first 200 of those models: 19 900 pairs, one warp per pair
    M = 200
    sub = coords[:M].contiguous()
    ap = clusco.clusco_gdt_allpairs(sub)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record(stream)
    clusco.clusco_gdt_allpairs(sub, ap)
    b.record(stream)
    torch.cuda.synchronize()
    ms_ap = a.elapsed_time(b)
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
