"""CPU-only checks: the C-ABI library builds for sm_100a, loads, and exports every symbol include/trimeg.h
declares (no compute call is made); the input generators are counter-based and reproducible; the N>1 host logic
(sharding + max-over-ranks timing) works under a world_size-2 gloo group."""
import ctypes
import os
import re
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_loads_and_exports_header_symbols():
    from paper_2606_24327_b200 import binding, build
    path = build.build()
    lib = ctypes.CDLL(path)
    header = open(os.path.join(ROOT, "include", "trimeg.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(trimeg_[a-z0-9_]+)\s*\(", header)))
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/trimeg.h but not exported"
    assert sorted(binding.EXPORTS) == declared
    # the binding wraps each C call under the same name (minus the prefix)
    for name in declared:
        short = name[len("trimeg_"):]
        if short in ("create", "destroy", "last_error"):
            continue
        assert hasattr(binding.Trimeg, short), short


def test_library_contains_only_sm100a_code():
    from paper_2606_24327_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_cpu_fallback_without_device():
    import torch
    from paper_2606_24327_b200.binding import Trimeg, TrimegError
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(TrimegError):
        Trimeg(0)


def test_product_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package (nor the C-ABI sources) may reference it."""
    pkg = os.path.join(ROOT, "paper_2606_24327_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "trimeg_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "trimeg_oracle.c")).read()
    assert "paper_2606_24327_b200" not in osrc.replace("paper_2606_24327_b200/csrc/", "").replace("never imports paper_2606_24327_b200", "")


def test_generators_are_counter_based():
    from paper_2606_24327_b200 import synth
    cfg = synth.CONFIGS[2]
    a = synth.make_markers(cfg, 1000, start=0)
    b = synth.make_markers(cfg, 400, start=600)
    for k in a:
        assert np.array_equal(a[k][600:], b[k]), k
    u = synth.uniform(7, 3, 200_000)
    assert 0 < u.min() and u.max() < 1 and abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 2e-3
    z = synth.normal(7, 3, 200_000)
    assert abs(z.mean()) < 1e-2 and abs(z.std() - 1) < 1e-2
    # first values are frozen: a change of the hash would silently change every workload
    assert np.allclose(synth.uniform(0, 0, 3), synth.uniform(0, 0, 5)[:3])
    RZ, tri = synth.make_mesh(synth.CONFIGS[1])
    assert tri.shape == (5040, 3) and RZ.shape == (29 * 90, 2)
    r = np.hypot(a["R"] - cfg.R0, a["Z"])
    assert r.min() >= 0.1 * cfg.a - 1e-12 and r.max() <= 0.9 * cfg.a + 1e-12
    assert (a["mu"] > 0).all() and (a["p"] == 1).all()


def test_field_dofs_are_consistent_derivatives():
    """The closed-form nodal derivatives handed to both sides are the derivatives of the closed-form value."""
    from paper_2606_24327_b200 import synth
    cfg = synth.CONFIGS[2]
    modes = synth.make_modes(cfg, 0)
    rng = np.random.default_rng(0)
    R = cfg.R0 + rng.uniform(-0.5, 0.5, 20) * cfg.a
    Z = rng.uniform(-0.5, 0.5, 20) * cfg.a
    ph = rng.uniform(0, 6, 20)
    h = 1e-5
    f = lambda r, z: synth.mode_field(modes, r, z, ph, cfg.R0, cfg.a)
    v = f(R, Z)
    fR = (f(R + h, Z) - f(R - h, Z)) / (2 * h)
    fZ = (f(R, Z + h) - f(R, Z - h)) / (2 * h)
    sc = np.abs(v[:, 1:3]).max()
    assert np.abs(fR[:, 0] - v[:, 1]).max() < 1e-6 * sc and np.abs(fZ[:, 0] - v[:, 2]).max() < 1e-6 * sc
    sc2 = np.abs(v[:, 3:]).max()
    assert np.abs(fR[:, 1] - v[:, 3]).max() < 1e-6 * sc2 and np.abs(fR[:, 2] - v[:, 4]).max() < 1e-6 * sc2
    assert np.abs(fZ[:, 2] - v[:, 5]).max() < 1e-6 * sc2 and np.abs(fZ[:, 1] - v[:, 4]).max() < 1e-6 * sc2


def test_shard_slices_partition_the_population():
    from paper_2606_24327_b200 import shard
    n, world = 1000, 4
    s = [shard.marker_slice(n, r, world) for r in range(world)]
    assert s[0][0] == 0 and all(s[i][1] == s[i + 1][0] for i in range(world - 1)) and s[-1][1] == n * world
    assert shard.job_rate(n, world, 2.0) == n * world / 2.0
    with pytest.raises(ValueError):
        shard.marker_slice(n, 4, 4)


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_2606_24327_b200 import shard, synth
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = synth.CONFIGS[1]
n = 5000
a, b = shard.marker_slice(n, rank, world)
m = synth.make_markers(cfg, b - a, a)
# each rank's slice equals the same slice of the single-process population
full = synth.make_markers(cfg, n * world, 0)
assert all(np.array_equal(m[k], full[k][a:b]) for k in m)
secs = shard.reduce_max_seconds(1.0 + rank, dist)
assert secs == float(world), secs
tot = torch.tensor([b - a], dtype=torch.int64)
dist.all_reduce(tot)
assert int(tot) == n * world
# the one collective of the path (SURVEY 8(e)): rank 0's field table reaches every rank through shard.broadcast_fields
class FakeBackend:
    def __init__(self, rank):
        self.table = (torch.arange(1000, dtype=torch.float64) * 0.5 if rank == 0 else torch.zeros(1000, dtype=torch.float64))
    def fields_export(self):
        return self.table.clone().view(torch.uint8)
    def fields_import(self, buf):
        self.table = buf.view(torch.float64).clone()
fb = FakeBackend(rank)
moved = shard.broadcast_fields(fb, dist, src=0)
assert moved == 8000 and torch.equal(fb.table, torch.arange(1000, dtype=torch.float64) * 0.5)
if rank == 0:
    print("RATE", shard.job_rate(n, world, secs))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_rank_gloo_sharding_and_timing(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(script), ROOT]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "RATE 5000.0" in r.stdout


def test_bench_gpus_2_spawns_two_ranks_and_reports_them():
    """`python bench.py --gpus 2` without a launcher must start its own two ranks (re-exec under torch.distributed.run on
    127.0.0.1) and print ONE line with n_gpus = 2; checked here on the reference arm (the oracle; needs no GPU)."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0",
           "--ref-markers", "500"]
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    import json
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
