"""Host side of the slab sharding (paper_1309_3859_b200/sharded.py), no GPU: partition arithmetic, shard / unshard
of the canonical link array with the ghost layers, and the one exchange of the path -- the all-gather and ordered
product of the per-shard slab products -- over torch.distributed with gloo, world size 2, on CPU tensors."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_partition_and_ghosts():
    from paper_1309_3859_b200 import sharded
    assert sharded.partition(64, 2, 4) == [(0, 16), (16, 16), (32, 16), (48, 16)]
    assert sharded.partition(12, 2, 4) == [(0, 4), (4, 4), (8, 2), (10, 2)]          # 6 slabs over 4 ranks
    assert sharded.partition(32, 4, 2) == [(0, 16), (16, 16)]
    assert sum(n for _, n in sharded.partition(24, 2, 5)) == 24
    for bad in ((10, 4, 2), (8, 2, 5), (8, 2, 0)):
        with pytest.raises(ValueError):
            sharded.partition(*bad)
    assert sharded.ghost_layers(16, 2) == 2 and sharded.ghost_layers(4, 4) == 4 and sharded.ghost_layers(3, 1) == 1
    assert sharded.ghost_layers(4, 1) == 2                                            # keeps the local extent even


def test_shard_unshard_round_trip_and_ghost_content():
    from paper_1309_3859_b200 import sharded
    Ns, Nt, d = 4, 12, 2
    rng = np.random.default_rng(1)
    links = rng.uniform(-3, 3, size=(4, Nt, Ns, Ns, Ns)).astype(np.float32)
    parts = sharded.partition(Nt, d, 3)
    shards = [sharded.shard_links(links, t0, n, d) for t0, n in parts]
    for s, (t0, n) in zip(shards, parts):
        assert s.shape[1] == n + 2
        assert np.array_equal(s[:, :n], links[:, t0:t0 + n])
        assert np.array_equal(s[:, n], links[:, (t0 + n) % Nt])                      # the next shard's frozen boundary layer
    assert np.array_equal(sharded.unshard_links(shards, parts), links)


WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_1309_3859_b200 import sharded
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
r = dist.get_rank()
rng = np.random.default_rng(7)                       # the same stream on both ranks: slab averages of a 3 x 4 x 6 x 64 problem
T = rng.standard_normal((3, 4, 6, 64)) + 1j * rng.standard_normal((3, 4, 6, 64))
parts = sharded.partition(12, 2, 2)                  # 6 slabs of thickness 2 -> 3 + 3
s0 = parts[r][0] // 2
local = torch.from_numpy(np.prod(T[:, :, s0:s0 + parts[r][1] // 2], axis=2))
got = sharded.gather_partial_products(local, dist)      # bytes only: the ordered product itself runs in libul (GPU tests)
ok = len(got) == 2 and all(np.array_equal(got[k].numpy(), np.prod(T[:, :, 3 * k:3 * k + 3], axis=2)) for k in range(2))
dist.barrier()
print("RESULT", r, bool(ok), tuple(got[0].shape))
dist.destroy_process_group()
"""


def test_exchange_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = 31500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    for r in range(2):
        line = [l for l in outs[r][0].splitlines() if l.startswith("RESULT")][0]
        assert line == f"RESULT {r} True (3, 4, 64)", line


def test_halo_ranges_and_shard_with_halo():
    from paper_1309_3859_b200 import sharded
    assert sharded.halo_ranges(8) == ((2, 4), (8, 10), (0, 2), (10, 12))
    with pytest.raises(ValueError):
        sharded.halo_ranges(1)
    Ns, Nt = 4, 12
    links = np.arange(4 * Nt * Ns ** 3, dtype=np.float32).reshape(4, Nt, Ns, Ns, Ns)
    s = sharded.shard_links_halo(links, 4, 4)
    assert s.shape[1] == 8 and np.array_equal(s[:, 2:6], links[:, 4:8])
    assert np.array_equal(s[:, :2], links[:, 2:4]) and np.array_equal(s[:, 6:], links[:, 8:10])
    s0 = sharded.shard_links_halo(links, 0, 4)
    assert np.array_equal(s0[:, :2], links[:, 10:12])                                  # periodic in t


HALO_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_1309_3859_b200 import sharded
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
r, nt_loc, GL = dist.get_rank(), 6, sharded.GL
# stand-in for the internal link view: [8 arrays][GL + nt_loc + GL layers][16 words]; own layers hold 1000 r + 10 arr + t
view = torch.full((8, nt_loc + 2 * GL, 16), -1, dtype=torch.int32)
for arr in range(8):
    for t in range(nt_loc):
        view[arr, GL + t] = 1000 * r + 10 * arr + t
sharded.exchange_halos(view, 5, nt_loc, dist, r, 2)
o = 1 - r
ok = all(int(view[5, t, 0]) == 1000 * o + 50 + (nt_loc - GL + t) for t in range(GL))                   # from below: the other rank's last layers
ok = ok and all(int(view[5, GL + nt_loc + t, 0]) == 1000 * o + 50 + t for t in range(GL))              # from above: its first layers
ok = ok and int(view[4, 0, 0]) == -1 and int(view[5, GL, 0]) == 1000 * r + 50                         # nothing else touched
dist.barrier()
print("RESULT", r, bool(ok))
dist.destroy_process_group()
"""


def test_halo_exchange_world_size_2_gloo(tmp_path):
    script = tmp_path / "halo_worker.py"
    script.write_text(HALO_WORKER.format(root=ROOT))
    port = 33500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    for r in range(2):
        line = [l for l in outs[r][0].splitlines() if l.startswith("RESULT")][0]
        assert line == f"RESULT {r} True", line
