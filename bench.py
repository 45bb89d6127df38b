#!/usr/bin/env python
"""Benchmark of the fused gather + RK4 marker push (BASELINE.json metric) on N B200s of one node.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--markers M] [--dt 0.05] [--impl reference]

One step = one RK4 step of the whole hot path over all markers of the config (store, periodic sort by cell,
locate, gather, equilibrium, equations of motion, weight, RK4 combine).  Prints ONE JSON line on rank 0.
`value` = marker RK4 pushes/s with the markers resident in HBM; `e2e` = the same through the C-ABI with HOST
buffers (H2D of the marker arrays and D2H of the result inside the timed region).
--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_24327_b200 import flopcount, shard, synth  # noqa: E402

METRIC = "marker RK4 pushes/sec incl. field gather (fp64, 1 B200), % of roofline"
UNIT = "marker-pushes/s"
# Algorithmic work: SURVEY.md 8(d)'s per-unit figure (943 flop per right-hand-side evaluation x 4 stages) is what the
# roofline uses; the count regenerated from this repo's own minimal formulation (paper_2606_24327_b200/flopcount.py,
# `python -m paper_2606_24327_b200.flopcount`) is printed beside it.
FLOP_PER_PUSH = 4.0 * flopcount.SURVEY_FLOP_PER_EVAL
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SM x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2
KEYS = ("R", "Z", "phi", "u", "w", "mu", "p")
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic.csv")   # dram bytes per launch of the dominant kernel, from a tracked ncu capture
ALGO_BYTES_PER_LAUNCH = 2 * 112 + 8 + 17   # per marker: 112 live record bytes in and out, permutation + key, one pass over the coefficient table
SORT_EVERY = 1                  # both phases re-bin every step (DESIGN.md section 6 "Sort interval": faster than BASELINE configs[2]'s every 10)
PARITY_TOL_10 = 1e-10           # north_star: marker state after 10 RK4 steps


def measured_traffic(cfg_name, n, variant):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, read from the tracked ncu summary
    profiles/traffic.csv (rows written from `ncu --set full` captures; each names the commit and the workload it was taken
    on; the last matching row wins).  None when no row is for this workload."""
    import csv
    best = (None, None)
    try:
        for r in csv.DictReader(open(TRAFFIC_FILE)):
            if r["workload"] == cfg_name and int(r["markers"]) == n and int(r["variant"]) == variant:
                best = (float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]), {k: r[k] for k in ("kernel", "commit", "source")})
    except Exception:
        pass
    return best


def make_inputs(cfg, n, start, pinned):
    """Markers [start, start+n) in chunks; returns dict of numpy arrays (views of pinned torch tensors if pinned)."""
    import torch
    host = {k: (torch.empty(n, dtype=torch.float64, pin_memory=True) if pinned else torch.empty(n, dtype=torch.float64)) for k in KEYS}
    views = {k: v.numpy() for k, v in host.items()}
    chunk = 2_000_000

    def fill(s):
        e = min(n, s + chunk)
        m = synth.make_markers(cfg, e - s, start + s)   # counter-based generator: any slice, any order
        for k in KEYS:
            views[k][s:e] = m[k]

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(32, os.cpu_count() or 8)) as ex:
        list(ex.map(fill, range(0, n, chunk)))
    return host, views


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True).start()
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None, "samples": len(sm), "reasons": sorted(reasons)}


def setup_case(cfg, backend):
    RZ, tri = synth.make_mesh(cfg)
    dphi, dap = synth.make_fields(cfg, RZ)
    backend.equilibrium_set(**synth.equilibrium_args(cfg))
    backend.species_set(**synth.species_args(cfg))
    backend.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    backend.fields_set(0, dphi)
    backend.fields_set(1, dap)
    return RZ, tri, (dphi, dap)


def time_oracle(cfg, n_sample, steps, start=0, oracle=None):
    """The oracle as it stands on the host cores: pushes/s on n_sample markers x steps RK4 steps."""
    from oracle import Oracle, oracle_threads
    o = oracle
    if o is None:
        o = Oracle()
        setup_case(cfg, o)
    m = synth.make_markers(cfg, n_sample, start)
    args = [m[k] for k in KEYS]
    t0 = time.perf_counter()
    o.push_rk4(*args, cfg.dt, steps)
    dt = time.perf_counter() - t0
    return n_sample * steps / dt, oracle_threads(), dt


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return
    n_sample = args.ref_markers
    from oracle import Oracle, oracle_threads
    o = Oracle()
    setup_case(cfg, o)
    m = synth.make_markers(cfg, n_sample, 0)
    st = [m[k] for k in KEYS]
    for _ in range(args.warmup):
        o.push_rk4(*[a[: max(1, n_sample // 10)] for a in st], cfg.dt, 1)
    t0 = time.perf_counter()
    cur = st
    for _ in range(args.steps):
        r = o.push_rk4(*cur, cfg.dt, 1)
        cur = [r[0], r[1], r[2], r[3], r[4], st[5], st[6]]
    el = time.perf_counter() - t0
    val = n_sample * args.steps / el
    sample = f"{n_sample} markers of {cfg.name} (of {cfg.n_markers}) per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(cfg, n_sample, args),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def _build_defs():
    try:
        from paper_2606_24327_b200.binding import build_info
        return build_info()
    except Exception:
        return None


def workload_config(cfg, n, args):
    return {"workload": f"{cfg.name}: {2 * cfg.nr * cfg.ntheta} triangles x {cfg.n_planes} planes, {n} markers/GPU, EM={cfg.em}, dt={cfg.dt}, RK4, sort every {args.sort_every} steps",
            "build_defs": _build_defs(), "markers_per_gpu": n, "triangles": 2 * cfg.nr * cfg.ntheta, "planes": cfg.n_planes, "dt": cfg.dt, "push_variant": args.variant, "sort_every": args.sort_every,
            "l2": "inputs_exceed_l2" if n * 104 > 126e6 else "l2_flushed_between_steps"}


def run_gather(args, cfg, n=None, steps=None, warmup=None):
    """BASELINE configs[4]: one field evaluation per point, points in random order and the same points sorted by cell, through
    trimeg_gather's staged path (the library bins the points itself, TMA-staged coefficient blocks) and through the direct
    one-thread-per-point kernel.  Returns the record ("mode": "gather"); not the headline metric (that is the push)."""
    import torch
    from paper_2606_24327_b200.binding import Trimeg
    n = n if n is not None else (args.markers if args.markers is not None else cfg.n_markers)
    steps = steps or args.steps
    warmup = args.warmup if warmup is None else warmup
    g = Trimeg(0)
    setup_case(cfg, g)
    host, views = make_inputs(cfg, n, 0, pinned=False)
    pts = {k: host[k].cuda() for k in ("R", "Z", "phi")}
    out = torch.empty((8, n), dtype=torch.float64, device="cuda")
    tri = torch.empty(n, dtype=torch.int32, device="cuda")

    def timed(P, mode):
        g.set_gather_mode(mode)
        for _ in range(warmup):
            g.gather(P["R"], P["Z"], P["phi"], out=out, tri_out=tri)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for s in range(steps):
            g.gather(P["R"], P["Z"], P["phi"], out=out, tri_out=tri)
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e-3 / steps, (g.gather_kernel_ms() if mode != 1 else None)

    t_rand_auto, parts_rand_auto = timed(pts, 0)
    t_rand, parts_rand = timed(pts, 2)
    t_rand_direct, _ = timed(pts, 1)
    # cell key = triangle x toroidal interval (caller numbering is enough to make the reads of a cell adjacent)
    k = torch.clamp((pts["phi"] % cfg.phi_period) / cfg.phi_period * cfg.n_planes, max=cfg.n_planes - 1).to(torch.int64)
    key = tri.to(torch.int64) * cfg.n_planes + k
    order = torch.argsort(key)
    spts = {q: v[order].contiguous() for q, v in pts.items()}
    del key, order, k
    t_sort_auto, parts_sort_auto = timed(spts, 0)
    t_sort, parts_sort = timed(spts, 2)
    t_sort_direct, _ = timed(spts, 1)
    T, Pn = 2 * cfg.nr * cfg.ntheta, cfg.n_planes
    table = T * Pn * 336
    algo = n * (24 + 4 + 64) + table          # points in, triangle id + 8 values out, one pass over the coefficient table
    peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"] if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else 6650.0
    line = {"mode": "gather", "metric": "field gathers/s (fp64, 1 B200)", "unit": "gathers/s", "n_gpus": 1, "steps": steps, "warmup": warmup,
            "value": n / t_rand_auto, "value_sorted_input": n / t_sort_auto, "dtype": "f64", "data": "synthetic",
            "ms": {"auto_unsorted_input": 1e3 * t_rand_auto, "auto_sorted_input": 1e3 * t_sort_auto, "staged_unsorted_input": 1e3 * t_rand, "staged_sorted_input": 1e3 * t_sort, "direct_unsorted_input": 1e3 * t_rand_direct,
                   "direct_sorted_input": 1e3 * t_sort_direct},
            "parts_ms": {"auto_unsorted_input": parts_rand_auto, "auto_sorted_input": parts_sort_auto, "staged_unsorted_input": parts_rand,
                         "staged_sorted_input": parts_sort},
            "config": {"workload": f"{cfg.name}: {T} triangles x {Pn} planes, {n} points, one evaluation of phi, A_par and gradients per point",
                       "l2": "inputs_exceed_l2", "build_defs": _build_defs()},
            "roofline": {"bound": "hbm", "achieved": algo / t_rand_auto / 1e9, "achieved_sorted_input": algo / t_sort_auto / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": algo / t_rand_auto / 1e9 / peak, "frac_sorted_input": algo / t_sort_auto / 1e9 / peak,
                         "frac_direct_unsorted_input": algo / t_rand_direct / 1e9 / peak, "traffic": None,
                         "kernel": "trimeg_gather, whole call in automatic mode (unsorted input: probe + k_gather_keys + scan + k_gather_scatter + k_gather_staged + k_gather_unsort; cell-sorted input: probe + k_gather_runs)",
                         "algorithmic_bytes": algo, "peak_kind": "MEASURED_PEAKS.json hbm_gbs" if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else "fallback"}}
    g.close()
    del pts, spts, out, tri
    torch.cuda.empty_cache()
    return line


def run_other_kernels(g, cfg, n, reps=3):
    """The per-marker calls beside the push (SURVEY.md 8(f) rows N2 / N3 and the paper's own kernel boundary, L89, L97-103) on the
    markers as the push left them (cell-ordered store), device buffers: milliseconds per call and the share of the HBM
    roofline for the bytes each must move (record in, result out).  Pullback last: it changes u and w."""
    import torch
    peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"] if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else 6650.0

    def timed(f):
        f()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            f()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    grid = 8 * 6 * cfg.n_planes * (cfg.nr + 1) * cfg.ntheta       # deposit: the DOF array written once
    calls = [("trimeg_rhs", lambda: g.rhs(), 128 + 40, 0), ("trimeg_density_g2p", lambda: g.density_g2p(0), 128 + 8, 0),
             ("trimeg_f_interp", lambda: g.f_interp(), 128 + 8, 0), ("trimeg_deposit", lambda: g.deposit(0), 128, grid),
             ("trimeg_pullback", lambda: g.pullback(), 256, 0)]
    rec = {"markers": n, "reps": reps, "hbm_peak_GBps": peak}
    for name, f, bytes_per_marker, extra in calls:
        ms = timed(f)
        algo = bytes_per_marker * n + extra
        rec[name] = {"ms": ms, "markers_per_s": n / (ms * 1e-3), "algorithmic_bytes": algo, "frac_hbm": algo / (ms * 1e-3) / 1e9 / peak}
    return rec


def run_push_extra(cfg, sort_every, steps=10, warmup=3, parity_n=2000):
    """One more BASELINE config through the same library on cuda:0 (device-resident, both phases' kernels, sort inside the
    timed region), with a small oracle sample; for the `other_configs` record of the bench line."""
    import torch
    from oracle import Oracle
    from paper_2606_24327_b200.binding import Trimeg
    g = Trimeg(0)
    setup_case(cfg, g)
    n = cfg.n_markers
    host, views = make_inputs(cfg, n, 0, pinned=False)
    dev = {k: v.cuda() for k, v in host.items()}
    g.set_push_variant(0)
    g.set_sort_interval(sort_every)
    g.markers_bind(*[dev[k] for k in KEYS])
    g.push_rk4(cfg.dt, warmup)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    g.push_rk4(cfg.dt, steps)
    b.record()
    torch.cuda.synchronize()
    sec = a.elapsed_time(b) * 1e-3
    st, km = g.push_stats(), g.push_kernel_ms()
    o = Oracle()
    setup_case(cfg, o)
    idx = np.unique(np.concatenate([np.arange(0, n, max(1, n // parity_n)), [n - 1]]))
    got = g.markers_get()
    tidx = torch.from_numpy(idx).cuda()
    got = {k: v[tidx].cpu().numpy() for k, v in got.items()}
    nst = warmup + steps
    exp = o.push_rk4(*[views[k][idx] for k in KEYS], cfg.dt, nst)
    errs = []
    for q, k in enumerate(("R", "Z", "phi", "u", "w")):
        dlt = np.abs(got[k] - exp[q])
        if k == "phi":
            dlt = np.minimum(dlt, np.abs(dlt - cfg.phi_period))
        errs.append(float(dlt.max() / max(np.abs(exp[q]).max(), 1e-300)))
    tol = PARITY_TOL_10 * max(1.0, (nst / 10.0) ** 2)
    evals = 4.0 * n - st["slow_path"] / steps
    rec = {"workload": f"{cfg.name}: {2 * cfg.nr * cfg.ntheta} triangles x {cfg.n_planes} planes, {n} markers, dt={cfg.dt}, sort every {sort_every} steps",
           "ms_per_step": 1e3 * sec / steps, "value": n * steps / sec, "unit": UNIT, "steps": steps, "warmup": warmup,
           "step_breakdown_ms": km, "retired_fraction_per_phase": st["retired"] / (2.0 * steps * n),
           "kernel_frac": (FLOP_PER_PUSH / 4.0) * evals / 2 / (km["push"] * 1e-3 / 2) / 1e12 / FP64_PEAK_TFLOPS,
           "whole_step_frac": FLOP_PER_PUSH * n / (sec / steps) / 1e12 / FP64_PEAK_TFLOPS,
           "parity": {"n": int(idx.shape[0]), "steps": nst, "max_rel": max(errs), "tol": tol,
                      "lost_set_equal": bool(((got["status"] != 0) == (exp[5] != 0)).all()), "ok": bool(max(errs) < tol)}}
    g.close()
    del dev, got
    torch.cuda.empty_cache()
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--markers", type=int, default=None, help="markers per GPU (default: the config's)")
    ap.add_argument("--dt", type=float, default=None)
    ap.add_argument("--variant", type=int, default=0, help="0 two-phase warp-specialised push, 1 simple")
    ap.add_argument("--sort-every", type=int, default=SORT_EVERY, help="re-sort the marker store every n RK4 steps (inside the timed region)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample", type=int, default=4_000_000, help="markers of the oracle cpu_baseline leg (x 4 steps)")
    ap.add_argument("--ref-markers", type=int, default=200_000, help="markers per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="skip the sampled oracle check of the timed run")
    ap.add_argument("--no-extras", action="store_true", help="skip the other BASELINE configs (1, 2 at both sort intervals, 4 gather) appended to the line")
    ap.add_argument("--parity-sample", type=int, default=10_000, help="markers of the timed run compared with the oracle")
    ap.add_argument("--gather", action="store_true", help="gather-only stress test (use with --config 4), unsorted vs cell-sorted points")
    args = ap.parse_args()

    import dataclasses
    cfg = synth.CONFIGS[args.config]
    if args.dt is not None:
        cfg = dataclasses.replace(cfg, dt=args.dt)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # no launcher: start the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1), same command line
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(1, args.gpus):
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU", file=sys.stderr)
        sys.exit(2)
    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
        return
    if args.gather:
        if rank == 0:
            print(json.dumps(run_gather(args, cfg)), flush=True)
        return

    import torch
    import torch.distributed as dist
    from paper_2606_24327_b200.binding import Trimeg

    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    n = args.markers if args.markers is not None else cfg.n_markers
    start, _ = shard.marker_slice(n, rank, world)

    g = Trimeg(local)
    fields_bcast = None
    if world > 1:
        # the one collective of the path: every rank loads the mesh, rank 0 alone turns the nodal DOFs into the
        # coefficient table, which is broadcast over NCCL (NCCL_DEBUG=INFO shows the transport: NVLink / NVLS)
        RZ, tri = synth.make_mesh(cfg)
        g.equilibrium_set(**synth.equilibrium_args(cfg))
        g.species_set(**synth.species_args(cfg))
        g.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
        if rank == 0:
            dphi, dap = synth.make_fields(cfg, RZ)
            g.fields_set(0, dphi)
            g.fields_set(1, dap)
        torch.cuda.synchronize()
        dist.barrier()
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b0.record()
        moved = shard.broadcast_fields(g, dist, src=0)
        b1.record()
        torch.cuda.synchronize()
        bsec = shard.reduce_max_seconds(b0.elapsed_time(b1) * 1e-3, dist)
        fields_bcast = {"bytes": moved, "ms": 1e3 * bsec, "GBps": moved / bsec / 1e9, "what": "export + dist.broadcast (NCCL) + import of the coefficient table"}
    else:
        setup_case(cfg, g)
    host, views = make_inputs(cfg, n, start, pinned=True)
    dev = {k: v.cuda(non_blocking=True) for k, v in host.items()}
    torch.cuda.synchronize()
    g.set_push_variant(args.variant)
    g.set_sort_interval(args.sort_every)
    g.markers_bind(*[dev[k] for k in KEYS])
    dfma = g.bench_dfma()
    dfma3 = g.bench_dfma_mix(1)     # DFMAs whose three operands are three different register pairs (2/3 of the pipe's rate: operand fetch)

    # ---- device-resident timing
    for _ in range(args.warmup):
        g.push_rk4(cfg.dt, 1)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    g.push_rk4(cfg.dt, args.steps)     # EXACTLY K steps, nothing else between the two events (no host round trip)
    ev1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None
    # counters and per-kernel times are read AFTER the timed region: launches, follow-up evaluations and retired markers of
    # the K steps; CUDA events recorded by the library on its own stream around each kernel group, mean over the K steps
    st = g.push_stats()
    km = g.push_kernel_ms()
    launches, slow, retired = st["launches"], st["slow_path"], st["retired"]
    total_s = shard.reduce_max_seconds(ev0.elapsed_time(ev1) * 1e-3, dist if world > 1 else None)
    value = shard.job_rate(n * args.steps, world, total_s)
    # dominant kernel: the phase kernel k_phase_ws, launched twice per step (phase A: k2, k3; phase B: k4, next k1).
    # Algorithmic flops per launch = 943 flop x the right-hand-side evaluations it performed (2 n minus those left to the
    # follow-up kernel), over its average launch duration from the library's CUDA events (sum of the two launches / 2).
    launches_per_step = 2 if args.variant == 0 else 1
    kern_s = km["push"] * 1e-3 / launches_per_step
    sort_ms, finish_ms = km["sort"], km["finish"]
    stage_evals = (4.0 * n - slow / args.steps) / launches_per_step
    achieved = (FLOP_PER_PUSH / 4.0) * stage_evals / kern_s / 1e12
    step_achieved = FLOP_PER_PUSH * n / (total_s / args.steps) / 1e12

    # ---- parity of THIS run: a strided sample of the markers just pushed (W + K steps) against the oracle on the same inputs
    parity, oracle_obj = None, None
    if not args.no_parity:
        from oracle import Oracle
        oracle_obj = Oracle()
        setup_case(cfg, oracle_obj)
        nst = args.warmup + args.steps
        idx = np.unique(np.concatenate([np.arange(0, n, max(1, n // args.parity_sample)), [n - 1]]))
        got = g.markers_get()
        tidx = torch.from_numpy(idx).cuda()
        got = {k: v[tidx].cpu().numpy() for k, v in got.items()}
        exp = oracle_obj.push_rk4(*[views[k][idx] for k in KEYS], cfg.dt, nst)
        tol = PARITY_TOL_10 * max(1.0, (nst / 10.0) ** 2)   # rounding-level differences grow at most quadratically over a few steps
        errs = {}
        for q, k in enumerate(("R", "Z", "phi", "u", "w")):
            dlt = np.abs(got[k] - exp[q])
            if k == "phi":
                dlt = np.minimum(dlt, np.abs(dlt - cfg.phi_period))
            errs["max_rel_" + k] = float(dlt.max() / max(np.abs(exp[q]).max(), 1e-300))
        lost_equal = bool(((got["status"] != 0) == (exp[5] != 0)).all())
        parity = {"n": int(idx.shape[0]), "steps": nst, "tol": tol, **errs, "lost_set_equal": lost_equal, "lost": int((exp[5] != 0).sum()),
                  "ok": bool(lost_equal and max(errs.values()) < tol), "against": "oracle/ (CPU, fp64) on the same seeded inputs"}
        del got, tidx

    # ---- end to end through the C-ABI with HOST buffers (pinned): H2D marker arrays, push, D2H result
    pinned_out = {k: torch.empty(n, dtype=torch.float64, pin_memory=True).numpy() for k in ("R", "Z", "phi", "u", "w")}
    pinned_out["status"] = torch.empty(n, dtype=torch.int32, pin_memory=True).numpy()
    e2e_steps = max(1, min(args.e2e_steps, args.steps))

    def e2e_step():
        g.markers_bind(*[views[k] for k in KEYS])
        g.push_rk4(cfg.dt, 1)
        g.markers_get(host=True, pinned=pinned_out)

    e2e_step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(e2e_steps):
        e2e_step()
    b.record()
    torch.cuda.synchronize()
    e2e_s = shard.reduce_max_seconds(a.elapsed_time(b) * 1e-3, dist if world > 1 else None)
    e2e_val = shard.job_rate(n * e2e_steps, world, e2e_s)
    traffic, traffic_src = measured_traffic(cfg.name, n, args.variant)
    own = flopcount.count()

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * total_s / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, n, args), "clocks": clocks,
                "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 7 * 8 * n, "d2h_bytes_per_step": (5 * 8 + 4) * n, "steps": e2e_steps,
                        "note": "every e2e step re-binds from HOST buffers, so it also pays the locate + k1 initialisation of a fresh store; PCIe-bound"},
                "gpu_launches": launches,
                "roofline": {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_PEAK_TFLOPS,
                             "traffic": traffic, "traffic_source": traffic_src,
                             "kernel": "k_phase_ws" if args.variant == 0 else "k_push_simple", "kernel_ms": 1e3 * kern_s,
                             "kernel_launches_per_step": launches_per_step,
                             "flop_per_push": FLOP_PER_PUSH, "stage_evals_per_launch": stage_evals,
                             "flop_count": {"used": "SURVEY.md 8(d): 943 flop per right-hand-side evaluation x 4",
                                            "regenerated_per_eval": own["total"]["flop"],
                                            "regenerated_parts": {k: v["flop"] for k, v in own.items() if k != "total"},
                                            "regenerated_ops": {k: own["total"][k] for k in ("add", "mul", "div", "sqrt", "exp")},
                                            "frac_with_regenerated_count": achieved / FP64_PEAK_TFLOPS * own["total"]["flop"] / flopcount.SURVEY_FLOP_PER_EVAL,
                                            "source": "python -m paper_2606_24327_b200.flopcount"},
                             "peak_kind": "nominal 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (derived, DESIGN.md)",
                             "measured_dfma_tflops": dfma, "frac_of_measured_dfma": achieved / dfma,
                             "measured_dfma_three_register_operands_tflops": dfma3,
                             "note_operands": "a DFMA with three different register-pair operands and no operand reuse issues every 3 cycles instead of 2 "
                                              "(trimeg_bench_dfma_mix; 235 of the ~610 FP64 instructions of an evaluation are of that kind): DESIGN.md section 6",
                             "whole_step_frac": step_achieved / FP64_PEAK_TFLOPS,
                             "hbm_algorithmic_GBps": ALGO_BYTES_PER_LAUNCH * n / kern_s / 1e9},
                "step_breakdown_ms": {"sort": sort_ms, "push": 1e3 * kern_s * launches_per_step, "finish": finish_ms},
                "slow_path_evals": slow, "retired_markers": retired, "parity": parity, "fields_bcast": fields_bcast}
        if not args.no_extras and world == 1 and args.config == 3 and n == cfg.n_markers:
            # the other BASELINE configs, same library, same run (not the headline)
            del pinned_out, host, views
            try:
                g.markers_bind(*[dev[k] for k in KEYS])
                g.push_rk4(cfg.dt, 2)
                line["other_kernels"] = run_other_kernels(g, cfg, n)
            except Exception as ex:
                line["other_kernels"] = {"error": repr(ex)}
            del dev
            g.close()
            torch.cuda.empty_cache()
            extras = {}
            try:
                extras["cfg1"] = run_push_extra(synth.CONFIGS[1], 1)
                extras["cfg2_sort_every_1"] = run_push_extra(synth.CONFIGS[2], 1)
                extras["cfg2_sort_every_10_as_BASELINE_states"] = run_push_extra(synth.CONFIGS[2], 10)
                extras["gather_cfg4"] = run_gather(args, synth.CONFIGS[4], n=synth.CONFIGS[4].n_markers, steps=3, warmup=1)
            except Exception as ex:   # the headline line must not be lost to an extra
                extras["error"] = repr(ex)
            line["other_configs"] = extras
        if not args.no_cpu_baseline:
            cpu_n = min(n, args.cpu_sample)
            v, cores, secs = time_oracle(cfg, cpu_n, 4, oracle=oracle_obj)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs,
                                    "sample": f"first {cpu_n} markers of the same workload x 4 RK4 steps"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    if parity is not None and not parity["ok"]:
        print(f"bench.py: parity against the oracle FAILED on rank {rank}: {parity}", file=sys.stderr)
        sys.exit(1)


if __name__ == "__main__":
    main()
