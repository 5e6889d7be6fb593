"""CPU-only checks: the C-ABI library loads and exports every symbol include/grpic.h
declares, the binding refuses to run without a GPU, input generators are deterministic, and
the particle-sharded multi-rank path (gloo, world_size 2) reproduces the unsharded deposit."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2503_04558_b200 import build as grpic_build
import inputs
from paper_2503_04558_b200 import sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_header_symbols():
    lib_path = grpic_build.build()
    lib = ctypes.CDLL(lib_path)
    header = open(os.path.join(ROOT, "include", "grpic.h")).read()
    names = sorted(set(re.findall(r"\b(grpic_[a-z_]+)\s*\(", header)))
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    lib.grpic_strerror.restype = ctypes.c_char_p
    assert lib.grpic_strerror(0) == b"ok"
    # argument errors are reported synchronously without a device
    assert lib.grpic_create(None, None) == -1
    assert lib.grpic_destroy(None) == -1


def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2503_04558_b200 import grpic
    with pytest.raises(grpic.GrpicError):
        grpic.Context(inputs.grid_params(16, 16, 0.5))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2503_04558_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "grpic_oracle" not in text, f


def test_inputs_deterministic_and_courant_values():
    a = inputs.config(1, nr=32, nth=32, n=1000)
    b = inputs.config(1, nr=32, nth=32, n=1000)
    for k in a["particles"]:
        assert np.array_equal(a["particles"][k], b["particles"][k])
    # SURVEY G16 values of 0.5 * Courant limit
    assert abs(inputs.courant_dt(inputs.grid_params(128, 128, 0.99)) - 1.0572e-2) < 2e-6
    assert abs(inputs.courant_dt(inputs.grid_params(1024, 1024, 0.99)) - 1.3010e-3) < 2e-7
    p = a["params"]
    ptc = a["particles"]
    m = inputs.kerr_schild(p["a"], 1.0, np.exp(ptc["x1"]), ptc["x2"])
    nrm = m["gu_rr"] * ptc["u1"] ** 2 + m["gu_thth"] * ptc["u2"] ** 2 + m["gu_phph"] * ptc["u3"] ** 2 \
        + 2 * m["gu_rph"] * ptc["u1"] * ptc["u3"]
    assert nrm.min() > 0.0099 and nrm.max() < 100.01        # |u| in [0.1, 10]


def test_shard_range_partitions():
    for n, w in [(10, 3), (7, 8), (100, 4), (0, 2)]:
        r = [sharding.shard_range(n, k, w) for k in range(w)]
        assert r[0][0] == 0 and r[-1][1] == n
        assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))


_WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import numpy as np, torch, torch.distributed as dist
import oracle
import inputs
from paper_2503_04558_b200 import sharding
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=int(sys.argv[1]), world_size=2)
cfg = inputs.config(1, nr=24, nth=20, n=600)
p, dt, ptc = cfg["params"], cfg["dt"], cfg["particles"]
lo, hi = sharding.shard_range(len(ptc["x1"]), dist.get_rank(), 2)
sub = {k: np.ascontiguousarray(v[lo:hi]) for k, v in ptc.items()}
new = oracle.push(p, cfg["fields"], sub, dt)
F = [torch.from_numpy(f) for f in oracle.deposit(p, sub, new, sub["w"], dt)]
sharding.allreduce_flux(F)
if dist.get_rank() == 0:
    newf = oracle.push(p, cfg["fields"], ptc, dt)
    Ff = oracle.deposit(p, ptc, newf, ptc["w"], dt)
    err = max(float(np.max(np.abs(a.numpy() - b))) / float(np.max(np.abs(b))) for a, b in zip(F, Ff))
    assert err < 1e-13, err
    print("OK", err)
dist.destroy_process_group()
"""


def test_particle_sharding_two_ranks_gloo(tmp_path):
    port = 29500 + os.getpid() % 2000
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % dict(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT) for r in range(2)]
    outs = [p.communicate(timeout=300)[0].decode() for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert "OK" in outs[0]


def test_bench_reference_arm_prints_contract_line():
    """`bench.py --impl reference` (the oracle timed on the host cores) prints one JSON line with the
    keys the driver reads; ranks other than 0 print nothing."""
    import json
    import subprocess
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
           "--warmup", "1", "--particles", "3000", "--grid", "64"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, check=True).stdout.strip().splitlines()
    d = json.loads(out[-1])
    assert d["impl"] == "reference" and d["unit"] == "particle-steps/s" and d["value"] > 0
    for k in ("metric", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["cpu_baseline"]["kind"] == "oracle"
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out1 = subprocess.run(cmd, capture_output=True, text=True, timeout=300, check=True, env=env).stdout.strip()
    assert out1 == ""


def test_bench_gpus_flag_starts_n_ranks_gloo():
    """`python bench.py --gpus 2` with no launcher in the environment starts the two ranks itself
    (torch.distributed.run on 127.0.0.1) and runs bench.py's OWN multi-rank host logic: rendezvous,
    per-rank seeds, ONE all-reduce of the contiguous 3-array flux block, max-time / sum-units
    aggregation, rank 0 alone printing the line (CPU stand-in with gloo)."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--host-logic-check"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                  # rank 1 prints nothing
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["ms_max"] == 11.0 and d["units_sum"] == 3000.0
    assert d["flux_sum"] == 3.0                             # (rank 0: 1) + (rank 1: 2), one collective
    assert d["seeds"] == [2, 2 + 7919] and d["shards"] == [501, 500]


def test_bench_relaunch_command_line():
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.relaunch_argv(["--gpus", "4", "--steps", "5"], 4, port=12345)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"]
    assert cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "12345"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "5"] and cmd[-5].endswith("bench.py")


def test_allreduce_flux_uses_one_collective_for_a_block(monkeypatch):
    """sharding.allreduce_flux on the contiguous [3, rows, pitch] block (or on its three views) issues
    exactly one all-reduce; three separate arrays fall back to three."""
    import torch
    import torch.distributed as dist
    calls = []
    monkeypatch.setattr(dist, "is_initialized", lambda: True)
    monkeypatch.setattr(dist, "get_world_size", lambda: 2)
    monkeypatch.setattr(dist, "all_reduce", lambda t, op=None: calls.append(t.numel()))
    block = torch.zeros(3, 4, 8, dtype=torch.float64)
    sharding.allreduce_flux(block)
    sharding.allreduce_flux(list(block.unbind(0)))
    assert calls == [96, 96]
    calls.clear()
    sharding.allreduce_flux([torch.zeros(4, 8) for _ in range(3)])
    assert calls == [32, 32, 32]


def test_bench_variant_option_and_guard_nodes():
    """bench.py --variant: the cubic-spline shape needs three guard nodes, so the workload of those
    variants is generated with ng = 3 (array shapes follow), the others with BASELINE's ng = 2; the
    option is parsed with the tuned kernel as default."""
    import bench
    assert bench.parse([]).variant == "cic-boris"
    for variant, ng in (("cic-vay", 2), ("spline3-boris", 3), ("spline3-vay", 3)):
        args = bench.parse(["--variant", variant, "--config", "1", "--grid", "24", "--particles", "50"])
        cfg = bench.workload(args, 0)
        p = cfg["params"]
        assert p["ng"] == ng and (p["nr"], p["nth"]) == (24, 24)
        assert all(f.shape == inputs.grid_shape(p) for f in cfg["fields"])
        assert len(cfg["particles"]["x1"]) == 50
        cfg1 = bench.workload(args, 1)            # another rank: same grid, its own particles
        assert cfg1["params"]["ng"] == ng and not np.array_equal(cfg1["particles"]["x1"], cfg["particles"]["x1"])
    with pytest.raises(SystemExit):
        bench.parse(["--variant", "spline5"])
