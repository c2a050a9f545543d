"""Host-side pieces of bench.py (no GPU): the max-over-ranks / sum-over-ranks aggregation on a world_size-2 gloo
group (replicas only, no collective on the data path), and the --impl reference arm."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
ms, units = bench.aggregate(10.0 + 5.0 * rank, 100.0 * (rank + 1))
dist.barrier()
dist.destroy_process_group()
print(json.dumps({{"rank": rank, "ms": ms, "units": units}}))
"""


def test_aggregate_takes_max_time_and_sums_units_over_two_gloo_ranks(tmp_path):
    port = 29000 + os.getpid() % 2000
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(os.environ, RANK=str(r), WORLD_SIZE="2"),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
        res = json.loads(o.strip().splitlines()[-1])
        assert res["ms"] == 15.0 and res["units"] == 300.0   # value = sum of units / max time on every rank


def test_aggregate_is_identity_without_a_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 7.0) == (3.5, 7.0)


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1",
                        "--warmup", "0", "--cpu-seconds", "0.2"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["dtype"] == "f64" and line["vs_baseline"] is None


def test_reference_arm_exits_quietly_on_other_ranks():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1"],
                       env=dict(os.environ, RANK="1", WORLD_SIZE="2"), capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
