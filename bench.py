#!/usr/bin/env python
"""bench.py -- GMMNLSE / MPA z-steps/s on B200 (BASELINE.json metric), one JSON line on stdout.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

A "step" is one ``gmmnlse_propagate`` call over ``LARGE_PER_STEP[config]`` MPA large steps (all §8(a)
rows: a1, a3-a11, every iteration, the convergence read-back) continuing from the previous step's
output field.  ``value`` = small z-steps per second with the field resident in HBM; ``e2e`` = the same
through ``gmmnlse_propagate_host`` (pinned staging, H2D + D2H inside the timed region).  N > 1 runs N
independent replicas (the path does not shard in this build: DESIGN.md "Multi-GPU"), one per rank.
``--impl reference`` times the fp64 CPU oracle (RK4IP) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "GMMNLSE z-steps/s (P modes, N samples, M planes)"
UNIT = "z-steps/s"
LARGE_PER_STEP = {1: 100, 2: 30, 3: 10, 4: 2, 5: 1}
ORACLE_MIN_SECONDS = 10.0             # the CPU sample runs whole RK4IP steps at the full (P, N) until this much time
ORACLE_MAX_STEPS = 400                 # ... or this many steps (configs 1-2 take milliseconds per step)
DEFAULT_CONFIG = 5


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sustained=d["bf16_tflops_sustained"],
                    source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i",
                 str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------ algorithmic work per launch
def algorithmic(kind, w, planes, a7_fused=False):
    """(bytes, flops) one launch of `kind` must move / execute for `planes` planes."""
    P, N = w.P, w.N
    Q = P * (P + 1) // 2
    c = 16 if w.precision else 8
    r = c // 2
    if kind in ("fft_to_time", "fft_to_freq"):
        return 3 * c * P * N * planes, 5 * N * np.log2(N) * P * planes      # in + table + out
    if kind == "pair_conv":
        return (c * P * N + r * Q * N) * planes, 0
    if kind == "contract":
        if a7_fused:                    # V in; A in and N_p out instead of U out (a7 runs in the epilogue)
            return (r * Q * N + 2 * c * P * N) * planes, (2.0 * Q * Q + 4.0 * P * P) * N * planes
        return 2 * r * Q * N * planes, 2.0 * Q * Q * N * planes
    if kind == "mode_reduce":
        return (r * Q * N + 2 * c * P * N) * planes, 4.0 * P * P * N * planes
    if kind == "scan":
        return 3 * c * P * N * planes, 0                                    # G in, psi old in, psi out
    return c * P * N * planes, 0


def max_over_ranks(ms: float, world: int, device) -> float:
    """Whole-job time of one timed region = the slowest rank's (contract: max over ranks)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_launch_field(A0, rank: int, seed_base: int):
    """Replica `rank` propagates the same fibre and pulse with its own seeded per-mode launch phases
    (rank 0: the configuration's own field); ranks share nothing on the data path."""
    if rank == 0:
        return A0
    rng = np.random.default_rng(seed_base + 1000 * rank)
    return (A0 * np.exp(2j * np.pi * rng.random((A0.shape[0], 1)))).astype(A0.dtype)


def job_value(world: int, z_steps_per_rank: int, ms_max_over_ranks: float) -> float:
    """Whole-job z-steps/s of `world` replicas: every rank advances its own field by z_steps_per_rank small steps in
    the slowest rank's time (weak scaling, no data-path collective)."""
    return world * z_steps_per_rank / (ms_max_over_ranks * 1e-3)


def run_launch_stub(args, stub_ms: float):
    """tests/test_bench_ranks.py only (GMMNLSE_BENCH_STUB_MS set): the N-rank launch of this script -- rendezvous,
    barrier, max over ranks, whole-job value, rank 0 printing -- with the measurement replaced by a fixed per-rank
    time, on CPU over gloo.  Nothing of the GPU path runs."""
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("gloo")
        dist.barrier()
    ms = max_over_ranks(stub_ms * (1 + rank), world, "cpu")
    z = args.steps * LARGE_PER_STEP[args.config] * 20
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": job_value(world, z, ms), "unit": UNIT, "n_gpus": world,
                          "steps": args.steps, "ms_per_step": ms / args.steps, "scaling": "weak", "stub": True}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_gpu(args):
    if os.environ.get("GMMNLSE_BENCH_STUB_MS"):
        return run_launch_stub(args, float(os.environ["GMMNLSE_BENCH_STUB_MS"]))
    import torch
    import torch.distributed as dist
    from paper_1708_05324_b200 import binding, workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the GPU path has no CPU fallback); use --impl reference")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.load_library()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def measure(cfg, K, Wm, with_events, host_path=False, seed_offset=0, contraction=None, stop_rule=0):
        w = workloads.make_config(cfg)
        n_large = LARGE_PER_STEP[cfg]
        L_step = n_large * w.M * w.dz
        cdt = np.complex128 if w.precision else np.complex64
        tdt = torch.complex128 if w.precision else torch.complex64
        A0 = w.A0.astype(cdt)
        A0 = replica_launch_field(A0, seed_offset, workloads.SEED_BASE)
        plan = binding.plan_from_workload(w, contraction=args.contraction if contraction is None else contraction,
                                          graph=1 if args.host_loop else 0, stop_rule=stop_rule)
        ckind, crank = plan.contraction_kind(), plan.lowrank_rank()
        stream = torch.cuda.current_stream()
        A = torch.from_numpy(A0).cuda()
        # e2e buffers: page-locked host memory (the library copies from / to it directly, no staging)
        h_a = torch.from_numpy(A0.copy()).pin_memory().numpy()
        h_b = torch.from_numpy(np.empty_like(A0)).pin_memory().numpy()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def step():
            nonlocal h_a, h_b
            if host_path:
                plan.propagate_host(h_a, L_step, h_b)
                h_a, h_b = h_b, h_a
            else:
                plan.propagate(A, L_step, A, stream)

        for _ in range(Wm):
            step()
        barrier()
        s0, l0 = plan.stats(), plan.launch_count()
        if with_events:
            plan.profile_enable(True)
        t0 = time.perf_counter()
        ev0.record(stream)
        for _ in range(K):
            step()
        ev1.record(stream)
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - t0) * 1e3
        dev_ms = ev0.elapsed_time(ev1)
        # propagate() syncs the stream at every convergence read-back, so host wall time and the
        # device-event span cover the same region; report the device span (max over ranks below)
        ms = max(dev_ms, 0.0) if not host_path else wall_ms
        prof = plan.profile_get() if with_events else None
        if with_events:
            plan.profile_enable(False)
        s1, l1 = plan.stats(), plan.launch_count()
        loop_kind = plan.loop_kind()
        barrier()
        ms = max_over_ranks(ms, world, "cuda")
        finite = bool(np.isfinite(h_a).all()) if host_path else bool(torch.isfinite(torch.view_as_real(A)).all())
        plan.destroy()
        it = s1["iterations"] - s0["iterations"]
        ls = s1["large_steps"] - s0["large_steps"]
        return dict(w=w, ms=ms, wall_ms=wall_ms, z_steps=K * n_large * w.M, iters=it, large=ls, prof=prof,
                    loop=loop_kind,
                    launches=l1 - l0, not_conv=s1["not_converged"] - s0["not_converged"], finite=finite,
                    bytes_io=int(A0.nbytes), ckind=ckind, crank=crank)

    def measure_sharded_world1(cfg, K, Wm, local):
        """paper_1708_05324_b200/sharded.py (host-driven loop, one all-gather + one max all-reduce per iteration over
        NCCL) with a process group of world size 1: what the exchange step and the host loop cost on one GPU against
        the device-side graph loop of `value`.  No scaling claim: this pool gives one GPU."""
        import socket
        from paper_1708_05324_b200 import sharded
        w = workloads.make_config(cfg)
        L_step = LARGE_PER_STEP[cfg] * w.M * w.dz
        A = torch.from_numpy(w.A0.astype(np.complex128 if w.precision else np.complex64)).cuda()
        own_group = not dist.is_initialized()
        if own_group:
            with socket.socket() as sk:
                sk.bind(("127.0.0.1", 0))
                port = sk.getsockname()[1]
            os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
        try:
            comm = sharded.TorchComm()
            plan = binding.plan_from_workload(w, graph=1)
            st = {}
            for _ in range(Wm):
                sharded.propagate_sharded(plan, comm, A, L_step, A, M=w.M, dz=w.dz, tol=w.tol)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(K):
                sharded.propagate_sharded(plan, comm, A, L_step, A, M=w.M, dz=w.dz, tol=w.tol, stats=st)
            torch.cuda.synchronize()
            ms = (time.perf_counter() - t0) * 1e3
            plan.destroy()
        finally:
            if own_group:
                dist.destroy_process_group()
        return {"value": round(K * LARGE_PER_STEP[cfg] * w.M / (ms * 1e-3), 2), "unit": UNIT, "ms_per_step": round(ms / K, 4),
                "iterations_per_large_step": round(st["iterations"] / max(st["large_steps"], 1), 3), "world_size": 1,
                "collectives_per_iteration": "all_gather of one [P][N] block + scalar max all_reduce (NCCL)"}

    cfg, K, Wm = args.config, args.steps, max(args.warmup, 3)
    peaks = _peaks()
    # `value`: the call a user makes (no per-kernel events; the MPA loop runs on the device as a CUDA graph).
    # `main`: the same region with the library's per-kernel CUDA events on (host loop), for the roofline object.
    with ClockSampler(local) as clk:
        plain = measure(cfg, K, Wm, with_events=False, seed_offset=rank)
        main = measure(cfg, K, Wm, with_events=True, seed_offset=rank)
    clocks = clk.summary()
    e2e = measure(cfg, K, Wm, with_events=False, host_path=True, seed_offset=rank)
    w = main["w"]
    value = job_value(world, plain["z_steps"], plain["ms"])

    # ---- roofline of the dominant kernel class, from the per-launch CUDA events of the timed region
    prof = {k: v for k, v in main["prof"].items() if v[1] > 0}
    dom = max(prof, key=lambda k: prof[k][0])
    tot_ms = sum(v[0] for v in prof.values())
    iters, large = main["iters"], main["large"]
    planes_total = {  # planes processed by all launches of a class over the region
        "fft_to_time": iters * w.M + large + K, "fft_to_freq": iters * w.M + large + K,
        "pair_conv": iters * w.M + large, "contract": iters * w.M + large, "mode_reduce": iters * w.M + large,
        "scan": iters * w.M, "advance": large, "misc": 0}
    shares = {}
    fused = "mode_reduce" not in prof
    for k, (ms_k, n_k) in prof.items():
        by, fl = algorithmic(k, w, planes_total.get(k, 0), fused)
        shares[k] = dict(ms=round(ms_k, 4), launches=n_k, share=round(ms_k / tot_ms, 4),
                         GBps=round(by / (ms_k * 1e-3) / 1e9, 1), TFLOPs=round(fl / (ms_k * 1e-3) / 1e12, 3))
    by, fl = algorithmic(dom, w, planes_total[dom], fused)
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")     # written from an ncu --set full capture
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        traffic = tj.get(f"cfg{cfg}", {}).get(dom)
        traffic_src = tj.get("_source", "profiles/traffic.json") + " (an earlier ncu --set full capture, replayed here: not measured by this run)"
    dom_ms, dom_n = prof[dom]
    if dom == "contract":
        # a6: `achieved` counts the method's useful packed-real flops (2 Q^2 N per plane).
        # The tcgen05 kernels reach fp32-grade accuracy by issuing three MMAs per product on hi/lo splits of the
        # operands, so the tensor pipe executes 3x the useful flops: `executed_*` reports that utilisation.
        # Peak: the measured bf16 sustained rate for the kind::f16 forms (fp16 = bf16 rate), x 0.5 (the guide's
        # nominal ratio) for the TF32 forms.
        ach = fl / (dom_ms * 1e-3) / 1e12
        ck = main["ckind"]
        # the timed region is a fraction of a second at full clock, so the BURST figure is the denominator of
        # `frac`; the sustained one is printed beside it
        if ck in (7, 8):
            kname, ratio, mult = "k_contract_h (a6, tcgen05 kind::f16 on fp16 hi/lo splits)", 1.0, 3
            pnote = f"peak = {peaks['source']} bf16 burst (fp16 runs at the bf16 rate)"
        elif ck in (3, 6):
            kname, ratio, mult = "k_contract_tc (a6, tcgen05 3xTF32)", 0.5, 3
            pnote = f"peak = {peaks['source']} bf16 burst x 0.5 (TF32 nominal ratio)"
        else:
            kname, ratio, mult = "k_contract (a6, fp32 FFMA)", 0.5, 1
            pnote = f"peak = {peaks['source']} bf16 burst x 0.5"
        peak, peak_s = peaks["bf16_burst"] * ratio, peaks["bf16_sustained"] * ratio
        roof = dict(bound="tensor", kernel=kname,
                    achieved=round(ach, 3), peak=round(peak, 1), unit="TFLOP/s", frac=round(ach / peak, 4),
                    peak_sustained=round(peak_s, 1), frac_of_sustained=round(ach / peak_s, 4),
                    traffic=traffic, traffic_source=traffic_src,
                    executed_tflops=round(mult * ach, 2),
                    executed_frac=round(mult * ach / peak, 4),
                    executed_frac_of_sustained=round(mult * ach / peak_s, 4),
                    note=f"useful flops 2*Q^2*N per plane; {pnote}; executed = {mult}x useful"
                         + (" (three MMAs per product: hi.lo, lo.hi, hi.hi)" if mult == 3 else ""))
    else:
        ach = by / (dom_ms * 1e-3) / 1e9
        roof = dict(bound="hbm", kernel=dom, achieved=round(ach, 1), peak=peaks["hbm"], unit="GB/s",
                    frac=round(ach / peaks["hbm"], 4), traffic=traffic, traffic_source=traffic_src,
                    note=f"algorithmic bytes / event-timed duration; peak = {peaks['source']} copy bandwidth")
    if main["ckind"] in (6, 8):
        roof["note"] += "; low-rank form selected: flop rates are dense-equivalent, not executed"
    roof["avg_launch_ms"] = round(dom_ms / dom_n, 4)
    roof["kernels"] = shares

    out = {
        "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": round(plain["ms"] / K, 4), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "c128" if w.precision else "c64 (f32)", "data": "synthetic",
        "config": {"workload": w.name, "baseline_config_index": cfg, "P": w.P, "N": w.N, "M": w.M,
                   "dz_m": w.dz, "z_steps_per_step": LARGE_PER_STEP[cfg] * w.M,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "working set per MPA iteration exceeds L2 (no flush)" if cfg >= 4 else
                         "working set is L2-resident by nature of the workload (no flush); not an HBM measurement"},
        "mode_sample_updates_per_s": round(value * w.P * w.N, 1),
        "iterations_per_large_step": round(plain["iters"] / max(plain["large"], 1), 3),
        "not_converged": plain["not_conv"], "finite": plain["finite"] and main["finite"],
        "ms_per_step_with_kernel_events": round(main["ms"] / K, 4),
        "e2e": {"value": round(job_value(world, e2e["z_steps"], e2e["ms"]), 2), "unit": UNIT,
                "h2d_bytes_per_step": e2e["bytes_io"], "d2h_bytes_per_step": e2e["bytes_io"] + (24 if e2e["loop"] == 1 else 8 * e2e["iters"] // K)},
        "gpu_launches": plain["launches"],
        "clocks": clocks, "roofline": roof,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = oracle_sample(cfg, 0, 0)
    out["config"]["contraction_kind"] = main["ckind"]
    out["config"]["a7"] = "in the contraction's epilogue (U never reaches HBM)" if fused else "separate kernel"
    out["config"]["mpa_loop"] = ("device (one CUDA graph per large step, WHILE node)" if plain["loop"] == 1
                                 else "host (read-back per iteration)")
    if rank == 0 and world == 1 and args.contraction == 0 and cfg >= 3 and not args.no_variants:
        # SURVEY.md 8(f) NEXT-4, reported beside the headline, never as it: the same propagation with the exact
        # low-rank form of the contraction (BASELINE.json names the dense one, which `value` measures)
        out["variants"] = {}
        try:
            lr = measure(cfg, K, Wm, with_events=False, contraction=8)
            out["variants"]["lowrank_contraction"] = {
                "value": round(lr["z_steps"] / (lr["ms"] * 1e-3), 2), "unit": UNIT, "rank": lr["crank"],
                "Q": w.P * (w.P + 1) // 2, "ms_per_step": round(lr["ms"] / K, 4), "contraction_kind": lr["ckind"],
                "iterations_per_large_step": round(lr["iters"] / max(lr["large"], 1), 3)}
        except binding.GmmnlseError as exc:
            out["variants"]["lowrank_contraction"] = {"unavailable": str(exc)}
        try:                                         # NEXT-4: the same dense product with S2's zero blocks skipped
            sp = measure(cfg, K, Wm, with_events=False, contraction=9)
            out["variants"]["block_sparse_contraction"] = {
                "value": round(sp["z_steps"] / (sp["ms"] * 1e-3), 2), "unit": UNIT, "ms_per_step": round(sp["ms"] / K, 4),
                "contraction_kind": sp["ckind"],
                "iterations_per_large_step": round(sp["iters"] / max(sp["large"], 1), 3)}
        except binding.GmmnlseError as exc:
            out["variants"]["block_sparse_contraction"] = {"unavailable": str(exc)}
        # reading S25: the a-posteriori stopping rule, same dense contraction; reported beside the headline
        # with its own iteration count (SURVEY.md reading S11/S12: variants of the iteration are allowed if both are)
        ap = measure(cfg, K, Wm, with_events=False, stop_rule=1)
        out["variants"]["aposteriori_stop_rule"] = {
            "value": round(ap["z_steps"] / (ap["ms"] * 1e-3), 2), "unit": UNIT, "ms_per_step": round(ap["ms"] / K, 4),
            "iterations_per_large_step": round(ap["iters"] / max(ap["large"], 1), 3), "not_converged": ap["not_conv"]}
        try:                                         # the plane-sharded driver, here on a world of ONE rank
            out["variants"]["plane_sharded_driver_world1"] = measure_sharded_world1(cfg, K, Wm, local)
        except Exception as exc:                     # (torch.distributed unavailable, port in use, ...)
            out["variants"]["plane_sharded_driver_world1"] = {"unavailable": str(exc)[:200]}
        try:                                         # the dense contraction on the 3xTF32 kernel (r01c-r01i's default)
            tf = measure(cfg, K, Wm, with_events=False, contraction=3)
            out["variants"]["tf32_contraction"] = {
                "value": round(tf["z_steps"] / (tf["ms"] * 1e-3), 2), "unit": UNIT,
                "ms_per_step": round(tf["ms"] / K, 4), "contraction_kind": tf["ckind"],
                "iterations_per_large_step": round(tf["iters"] / max(tf["large"], 1), 3)}
        except binding.GmmnlseError as exc:
            out["variants"]["tf32_contraction"] = {"unavailable": str(exc)}
    if rank == 0 and args.all_configs and world == 1:
        others = []
        for c in (1, 2, 3, 4):
            if c == cfg:
                continue
            m = measure(c, 10, 3, with_events=False)
            others.append({"workload": m["w"].name, "z_steps_per_s": round(m["z_steps"] / (m["ms"] * 1e-3), 1),
                           "ms_per_step": round(m["ms"] / 10, 4), "z_steps_per_step": LARGE_PER_STEP[c] * m["w"].M,
                           "iterations_per_large_step": round(m["iters"] / max(m["large"], 1), 3),
                           "mpa_loop": "device" if m["loop"] == 1 else "host"})
        out["other_workloads"] = others
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------ M-sweep (Fig. 3 shape)
def run_sweep(args):
    """the paper's one performance experiment (Fig. 3) has a serial
    integrator on the GPU against the MPA for several M on a 10-mode GRIN fibre with z_nl/dz ~ 200.  The
    figure's bars are not available; this prints the same comparison for this implementation: the serial
    RK4IP (gmmnlse_propagate_rk4ip) and the MPA at each M, same fibre, pulse, dz and length."""
    import torch
    from paper_1708_05324_b200 import binding, workloads
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep-M: no CUDA device")
    binding.load_library()
    w = workloads.make_config(3, max_group=3)                     # 10-mode GRIN, 200 kW, 300 fs, N = 8192
    gamma = w.kappa * w.S[0, 0, 0, 0]
    z_nl = 1.0 / (gamma * w.meta.get("p_peak", 200e3))
    w.dz = z_nl / 200.0
    n_small = 400
    L = n_small * w.dz
    A = torch.from_numpy(w.A0.astype(np.complex64)).cuda()
    stream = torch.cuda.current_stream()

    def timed(fn, reps=3):
        fn(); torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    out_rk = torch.empty_like(A)
    g = 1 if args.host_loop else 0
    with binding.plan_from_workload(w, M=1, graph=g) as plan:
        ms = timed(lambda: plan.propagate_rk4ip(A, L, out_rk, stream))
    ref = out_rk.cpu().numpy().astype(np.complex128)
    res = {"sweep": "fig3-like", "workload": "10-mode GRIN (config-3 fibre, groups 0-3), N=8192, 200 kW 300 fs, "
                                             "Kerr+Raman+shock", "P": w.P, "N": w.N, "dz_m": w.dz,
           "z_nl_over_dz": 200.0, "small_steps": n_small, "unit": UNIT,
           "loops": "host (options.graph = 1)" if g else "device (CUDA graphs: MPA WHILE loop, replayed RK4IP step)",
           "serial_rk4ip": {"z_steps_per_s": round(n_small / (ms * 1e-3), 1), "ms": round(ms, 3),
                            "nonlinear_evals_per_step": 4}, "mpa": []}
    for M in (1, 2, 4, 5, 10, 20, 40):
        out = torch.empty_like(A)
        with binding.plan_from_workload(w, M=M, graph=g) as plan:
            ms = timed(lambda: plan.propagate(A, L, out, stream))
            s0 = plan.stats()
            plan.propagate(A, L, out, stream); torch.cuda.synchronize()
            s1 = plan.stats()
        o = out.cpu().numpy().astype(np.complex128)
        res["mpa"].append({"M": M, "z_steps_per_s": round(n_small / (ms * 1e-3), 1), "ms": round(ms, 3),
                           "iterations_per_large_step": round((s1["iterations"] - s0["iterations"])
                                                              / max(s1["large_steps"] - s0["large_steps"], 1), 2),
                           "rel_l2_vs_serial": float(np.linalg.norm(o - ref) / np.linalg.norm(ref))})
    best = max(res["mpa"], key=lambda r: r["z_steps_per_s"])
    res["best_M"] = best["M"]
    res["mpa_over_serial"] = round(best["z_steps_per_s"] / res["serial_rk4ip"]["z_steps_per_s"], 2)
    print(json.dumps(res))


# ------------------------------------------------------------------------------ oracle (CPU) leg
def cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(cfg, K, Wm):
    """Time the fp64 oracle as it stands (oracle/gmmnlse_oracle.py) at the configuration's FULL (P, N): one
    nonlinear-operator evaluation (O2), then whole RK4IP small steps (O3, 4 evaluations each).  K > 0: exactly K
    timed steps after Wm warm-up steps (the --impl reference arm); K == 0: as many steps as it takes to pass
    ORACLE_MIN_SECONDS (at least one).  Nothing is extrapolated: value = steps done / seconds taken."""
    from oracle import gmmnlse_oracle as O
    from paper_1708_05324_b200 import workloads
    w = workloads.make_config(cfg)
    omega = O.omega_grid(w.N, w.dt)
    D = O.dispersion_operator(w.beta, omega)
    nl = lambda X: O.nonlinear_op_freq(X, w.S, w.kappa, omega, w.omega0, w.f_R, w.h_R, w.dt, w.shock)
    t0 = time.perf_counter()
    O.nonlinear_op(w.A0, w.S, w.kappa, w.omega0, w.f_R, w.h_R, w.dt, w.shock)
    op_sec = time.perf_counter() - t0
    At = O.to_freq(w.A0)
    for _ in range(Wm):
        At = O.rk4ip_step(At, w.dz, D, nl)
    done, step_secs = 0, []
    t0 = time.perf_counter()
    while True:
        t1 = time.perf_counter()
        At = O.rk4ip_step(At, w.dz, D, nl)
        step_secs.append(time.perf_counter() - t1)
        done += 1
        if (K > 0 and done >= K) or (K == 0 and (time.perf_counter() - t0 >= ORACLE_MIN_SECONDS
                                                   or done >= ORACLE_MAX_STEPS)):
            break
    sec = time.perf_counter() - t0
    try:
        import threadpoolctl
        cores = max([p["num_threads"] for p in threadpoolctl.threadpool_info()] or [1])
    except Exception:
        cores = os.cpu_count() or 1
    return {"value": round(done / sec, 5), "unit": UNIT, "cores": cores, "cpu_model": cpu_model(),
            "host_cpus": os.cpu_count(), "kind": "oracle",
            "sample": f"{done} RK4IP small step(s) (4 nonlinear-operator evaluations each) of {w.name} at its full "
                      f"shape P={w.P}, N={w.N}: {sec:.1f} s; one nonlinear-operator evaluation alone: {op_sec:.2f} s",
            "steps": done, "seconds": round(sec, 2), "ms_per_rk4ip_step": round(1e3 * float(np.mean(step_secs)), 1),
            "nonlinear_op_evals_per_s": round(1.0 / op_sec, 4),
            "finite": bool(np.isfinite(At).all())}


def run_reference(args):
    """The reference arm of this tier is the oracle: one "step" = one RK4IP small step (dz) at the full shape, so
    value = steps / seconds is the same z-steps/s metric and ms_per_step x steps is the time the timed loop took."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1708_05324_b200 import workloads
    w = workloads.make_config(args.config)
    # bound the run to a few minutes: one probe step sets the cap on the timed steps
    t0 = time.perf_counter()
    probe = oracle_sample(args.config, 1, 0)
    per_step = probe["seconds"]
    K = max(1, min(args.steps, int(150.0 / max(per_step, 1e-3))))
    Wm = min(args.warmup, 1 if per_step > 1.0 else 3)
    cb = oracle_sample(args.config, K, Wm)
    out = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT,
           "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": K, "warmup": Wm,
           "ms_per_step": round(1e3 * cb["seconds"] / K, 1),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128 (f64)",
           "data": "synthetic",
           "config": {"workload": w.name, "baseline_config_index": args.config, "P": w.P, "N": w.N, "M": w.M,
                      "dz_m": w.dz, "integrator": "RK4IP (oracle O3), fixed step dz", "z_steps_per_step": 1,
                      "steps_requested": args.steps, "steps_run": K,
                      "note": "a step is one RK4IP small step at the full shape; the step count is capped so the run "
                              "ends within a few minutes"},
           "cpu_baseline": cb,
           "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "wall_s": round(time.perf_counter() - t0, 1)}
    print(json.dumps(out))


def spawn_ranks(n: int) -> int:
    """`python bench.py --gpus N` outside torchrun: start the N ranks ourselves, exactly the way the driver would
    (one process per GPU, NCCL rendezvous on 127.0.0.1), and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="graft", choices=["graft", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--all-configs", action="store_true", help="also time configs 1-4 briefly (other_workloads)")
    ap.add_argument("--host-loop", action="store_true",
                    help="options.graph = 1: take the MPA convergence decision on the host (read-back per iteration) "
                         "instead of in the CUDA-graph WHILE loop")
    ap.add_argument("--contraction", type=int, default=0,
                    help="options.contraction for every measurement (0 auto = the dense kind::f16 tcgen05 form; 3 dense 3xTF32; "
                         "6 / 8 low-rank on the TF32 / f16 kernel)")
    ap.add_argument("--no-variants", action="store_true", help="skip the low-rank variant measurement")
    ap.add_argument("--sweep-M", action="store_true", help="serial RK4IP vs MPA(M) on a 10-mode GRIN (Fig. 3 shape)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "graft" and not args.sweep_M:
        raise SystemExit(spawn_ranks(args.gpus))
    if args.sweep_M:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
