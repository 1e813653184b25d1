"""Static multi-GPU partition: host-side logic on CPU.

The shard bookkeeping is checked directly, and the N > 1 exchange (forces in / state out) with
world_size 2 on `gloo`, the CUDA solver replaced by a stand-in that has no arithmetic of the method
(x += dt v; v += dt F) - what is under test is which rank gets which cell and where it lands."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1911_03062_b200.partition import Partition, static_partition

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_static_partition_is_even_disjoint_and_contiguous_per_type(world):
    rng = np.random.default_rng(3)
    toc = rng.choice(3, size=1001, p=[0.85, 0.1, 0.05]).astype(np.int32)
    parts = static_partition(toc, world)
    allc = np.concatenate(parts)
    assert np.array_equal(np.sort(allc), np.arange(toc.shape[0]))            # disjoint cover
    sizes = [p.shape[0] for p in parts]
    assert max(sizes) - min(sizes) <= 1                                      # totals balanced
    for t in range(3):
        ids_t = np.flatnonzero(toc == t)
        per_rank = [p[toc[p] == t] for p in parts]
        counts = [q.shape[0] for q in per_rank]
        assert max(counts) - min(counts) <= 1                                # every type balanced
        for q in per_rank:                                                   # one contiguous range of the type's cells
            if q.shape[0]:
                pos = np.searchsorted(ids_t, q)
                assert np.array_equal(pos, np.arange(pos[0], pos[0] + q.shape[0]))


def test_partition_more_ranks_than_cells_and_empty():
    parts = static_partition(np.array([0, 1, 0], dtype=np.int32), 8)
    assert sorted(int(i) for p in parts for i in p) == [0, 1, 2] and max(p.shape[0] for p in parts) == 1
    assert all(p.shape[0] == 0 for p in static_partition(np.zeros(0, dtype=np.int32), 2))
    with pytest.raises(ValueError):
        static_partition(np.zeros(4, dtype=np.int32), 0)


def test_scatter_assemble_round_trip_mixed_types():
    toc = np.array([0, 1, 1, 0, 2, 0, 1], dtype=np.int32)
    nv = [5, 3, 7]
    part = Partition(toc, nv, 3)
    total = 3 * sum(nv[t] for t in toc)
    glob = np.arange(total, dtype=np.float64)
    pieces = [part.scatter(glob, r) for r in range(3)]
    assert sum(p.shape[0] for p in pieces) == total and [p.shape[0] for p in pieces] == part.counts
    assert np.array_equal(part.assemble(pieces), glob)
    # a rank's buffer is its cells back to back, each [n][3], in ascending cell id
    r = 1
    expect = np.concatenate([glob[part.cell_off[c]:part.cell_off[c + 1]] for c in part.cell_ids[r]])
    assert np.array_equal(pieces[r], expect)


_WORKER = r"""
import sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch.distributed as dist
from paper_1911_03062_b200.partition import ShardedSolver

class CT:
    def __init__(self, n): self.rest_positions = np.zeros((n, 3))

class StandIn:                                   # explicit Euler on free particles: no method arithmetic
    def __init__(self, cell_types, toc, dt): self.dt = dt
    def set_state(self, x, v=None): self.x = x.copy(); self.v = np.zeros_like(x) if v is None else v.copy()
    def set_forces(self, f): self.f = f.copy()
    def step(self, k):
        self.x = self.x + self.dt * self.v; self.v = self.v + self.dt * self.f
    def get_state(self, dtype="fp64", where="host"): return self.x, self.v

rank = int(sys.argv[1])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
types = [CT(6), CT(4)]
toc = np.array([0, 1, 0, 0, 1, 0, 0], dtype=np.int32)
n = 3 * sum(types[t].rest_positions.shape[0] for t in toc)
rng = np.random.default_rng(0)                   # same global buffers on every rank
x0, v0, f = rng.normal(size=n), rng.normal(size=n), rng.normal(size=n)
s = ShardedSolver(types, toc, 0.5, rank, 2, solver_factory=StandIn)
s.set_state(x0, v0); s.set_forces(f); s.step(1); s.step(1)
x, v = s.gather_state()
ex = x0 + 0.5 * v0 + 0.5 * (v0 + 0.5 * f); ev = (v0 + 0.5 * f) + 0.5 * f
print(json.dumps({{"rank": rank, "ok": bool(np.array_equal(x, ex) and np.array_equal(v, ev)),
                  "cells": [int(c) for c in s.cell_ids]}}))
dist.destroy_process_group()
"""


def test_sharded_solver_gather_gloo_world2(tmp_path):
    import json
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (_, err) in zip(procs, outs):
        assert p.returncode == 0, err
    rows = [json.loads(out.strip().splitlines()[-1]) for out, _ in outs]
    assert all(r["ok"] for r in rows)
    assert sorted(rows[0]["cells"] + rows[1]["cells"]) == list(range(7))
