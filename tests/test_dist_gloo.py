"""CPU test (gloo, world_size 2) of the N>1 host logic bench.py uses: rendezvous on 127.0.0.1,
barriers, max-over-ranks of the device time, whole-job aggregate (replicas, weak scaling)."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
from paper_2503_22139_b200.dist import Ranks, whole_job_rate
r = Ranks(backend="gloo")
r.barrier()
ms_total = 100.0 if r.rank == 0 else 250.0           # rank 1 is the slow replica
value, ms_step = whole_job_rate(1000.0 * (r.rank + 1), r, ms_total, steps=10)
mx = r.max_over_ranks(r.rank * 7.0)
r.close()
print(json.dumps({"rank": r.rank, "world": r.world, "value": value, "ms_step": ms_step, "mx": mx}))
"""


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_rank_gloo_max_time_and_aggregate():
    import json
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=120)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["world"] == 2
        assert o["ms_step"] == 25.0                      # max over ranks (250 ms / 10 steps)
        assert abs(o["value"] - 3000.0 / 0.025) < 1e-6   # all ranks' units / max time
        assert o["mx"] == 7.0


def test_single_process_needs_no_process_group():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_2503_22139_b200.dist import Ranks, whole_job_rate\n"
            "r = Ranks(backend='gloo'); v, ms = whole_job_rate(500.0, r, 50.0, 5); r.close(); print(v, ms)") % ROOT
    out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr[-2000:]
    v, ms = out.stdout.split()
    assert float(ms) == 10.0 and abs(float(v) - 50000.0) < 1e-9


# ------------------------------------------------------------------ z-slab sharding
def test_slab_bounds_partition_every_layer_exactly_once():
    sys.path.insert(0, ROOT)
    from paper_2503_22139_b200.dist import slab_bounds
    for nbz in (0, 1, 3, 8, 16, 32, 33):
        for world in (1, 2, 3, 4, 8, 16):
            cover = []
            sizes = []
            for r in range(world):
                lo, hi = slab_bounds(nbz, r, world)
                assert 0 <= lo <= hi <= nbz
                cover += list(range(lo, hi)); sizes.append(hi - lo)
            assert cover == list(range(nbz))                 # contiguous, ordered, no gap, no overlap
            assert max(sizes) - min(sizes) <= 1              # balanced
    import pytest
    with pytest.raises(ValueError):
        slab_bounds(4, 2, 2)


SLAB_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch
from paper_2503_22139_b200.dist import Ranks, slab_bounds, sharded_backward

class FakePlan:                       # host-side stand-in: the accumulate / all-reduce / finish protocol
    def __init__(self, rank): self.acc = torch.full((6, 12), float(rank + 1)); self.calls = []
    def backward_accumulate(self, w, g): self.calls.append("acc")
    def accumulators(self, ch): self.calls.append("view%%d" %% ch); return self.acc.view(-1)
    def backward_finish(self, ch, grads=None): self.calls.append("fin"); return self.acc.clone()

r = Ranks(backend="gloo")
lo, hi = slab_bounds(5, r.rank, r.world)
plan = FakePlan(r.rank)
out = sharded_backward(plan, torch.zeros(6, 1), None, r)
r.close()
print(json.dumps({"rank": r.rank, "slab": [lo, hi], "calls": plan.calls, "sum": float(out[0, 0])}))
"""


def test_two_rank_gloo_sharded_backward_all_reduces_between_the_halves():
    import json
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", SLAB_WORKER % ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=120)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    assert outs[0]["slab"] == [0, 3] and outs[1]["slab"] == [3, 5]
    for o in outs:
        assert o["calls"] == ["acc", "view1", "fin"]
        assert o["sum"] == 3.0                               # 1 + 2: summed over both ranks before a5


BATCH_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch
from paper_2503_22139_b200.dist import Ranks, batch_bounds, all_reduce_grads
r = Ranks(backend="gloo")
lo, hi = batch_bounds(8, r.rank, r.world)
g = [torch.full((5, 3), float(hi - lo)), torch.full((5,), float(r.rank + 1))]       # partial gradients of shared parameters
all_reduce_grads(g, r)
r.close()
print(json.dumps({"rank": r.rank, "b": [lo, hi], "g0": float(g[0][0, 0]), "g1": float(g[1][0])}))
"""


def test_two_rank_gloo_projection_batch_sharding_and_gradient_sum():
    import json
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", BATCH_WORKER % ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=120)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    assert outs[0]["b"] == [0, 4] and outs[1]["b"] == [4, 8]
    for o in outs:
        assert o["g0"] == 8.0 and o["g1"] == 3.0             # sums over both ranks


def test_slab_bounds_by_keys_partition_and_balance():
    """Key-balanced cuts: every layer owned exactly once, contiguous; no slab holds more than total/world plus one
    layer's keys; equal weights give the equal-layer split; a clustered profile moves the cuts into the cluster."""
    sys.path.insert(0, ROOT)
    import numpy as np
    from paper_2503_22139_b200.dist import slab_bounds, slab_bounds_by_keys
    rng = np.random.default_rng(5)
    profiles = [[1] * 32, [0] * 8, [5], list(rng.integers(0, 1000, 32)), [0, 0, 0, 900, 50, 50, 0, 0],
                list((1000 * np.exp(-0.5 * ((np.arange(32) - 12) / 3.0) ** 2)).astype(int))]
    for w in profiles:
        for world in (1, 2, 3, 4, 8):
            cover, loads = [], []
            for r in range(world):
                lo, hi = slab_bounds_by_keys(w, r, world)
                assert 0 <= lo <= hi <= len(w)
                cover += list(range(lo, hi)); loads.append(sum(w[lo:hi]))
            assert cover == list(range(len(w)))
            if sum(w) > 0:
                assert max(loads) <= sum(w) / world + max(w) + 1e-9
    for world in (1, 2, 4, 8):
        for r in range(world):
            assert slab_bounds_by_keys([7] * 32, r, world) == slab_bounds(32, r, world)
    # the Gaussian-shaped profile: equal layers would give rank 0 of 4 the layers 0..7 (few keys); key balance does not
    w = profiles[-1]
    eq = [sum(w[slab_bounds(32, r, 4)[0]:slab_bounds(32, r, 4)[1]]) for r in range(4)]
    kb = [sum(w[slab_bounds_by_keys(w, r, 4)[0]:slab_bounds_by_keys(w, r, 4)[1]]) for r in range(4)]
    assert max(kb) < 0.6 * max(eq)
