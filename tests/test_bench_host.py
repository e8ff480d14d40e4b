"""Host-side logic of bench.py that needs no GPU: the step's update count, the per-rank seeds of the
N > 1 replicas, the max-over-ranks reduction (world size 2, gloo, on CPU) and the reference arm's line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_updates_per_step_matches_survey_counts():
    sys.path.insert(0, ROOT)
    import bench
    w = dict(bench.WORKLOAD)
    V = w["Ns"] ** 3 * w["Nt"]
    total, full, masked = bench.updates_per_step(w)
    sweeps = w["n_hb"] + w["n_or"]
    assert full == sweeps * 4 * V                                   # 4V links per full sweep
    assert masked == sweeps * (V + 3 * V // 2)                      # d = 2: V temporal + 3V/2 spatial (S8(a) a6: 2.5 V)
    assert total == full + w["n_sub"] * masked
    assert bench.rank_seed(5, 0) == 5 and bench.rank_seed(5, 3) == 8


WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
r = dist.get_rank()
m = bench.distributed_max(10.0 + 5.0 * r, dist)
seeds = [None, None]
dist.all_gather_object(seeds, bench.rank_seed(5, r))
dist.barrier()
if r == 0:
    print("RESULT", m, seeds)
dist.destroy_process_group()
"""


def test_max_over_ranks_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = 29500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = [l for l in outs[0][0].splitlines() if l.startswith("RESULT")][0]
    assert line == "RESULT 15.0 [5, 6]"                             # max over ranks; independent seeds per rank


@pytest.mark.timeout(300)
def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--sample-ns", "32"], capture_output=True, text=True, timeout=280)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "link_updates_per_s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
