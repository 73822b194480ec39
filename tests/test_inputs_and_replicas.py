"""Seeded input generators (structure of the BASELINE.json configs) and the N>1 replica path on CPU (gloo)."""
import os
import subprocess
import sys
from pathlib import Path

import numpy as np

from paper_2106_03452_b200 import inputs

ROOT = Path(__file__).resolve().parents[1]


def test_generators_are_seeded_and_in_the_unit_cube():
    for shape, P in [("sphere", 3000), ("torus", 5000), ("ellipsoids3", 4000), ("ellipsoids8", 4000), ("bumpy", 5000)]:
        a = inputs.make_cloud(shape, P, seed=4)
        b = inputs.make_cloud(shape, P, seed=4)
        c = inputs.make_cloud(shape, P, seed=5)
        assert a[0].dtype == np.float32 and a[0].shape == (P, 3) and a[1].shape == (P, 3)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and not np.array_equal(a[0], c[0])
        assert a[0].min() >= 0.0 and a[0].max() < 1.0
        assert np.abs(np.linalg.norm(a[1], axis=1) - 1.0).max() < 1e-5


def test_surface_structure():
    c, n = inputs.make_cloud("sphere", 3000)
    assert np.abs(np.linalg.norm(c - 0.5, axis=1) - 0.3).max() < 1e-6
    assert np.abs(n - (c - 0.5) / 0.3).max() < 1e-5
    c, n = inputs.make_cloud("torus", 20000)
    ring = np.hypot(c[:, 0] - 0.5, c[:, 1] - 0.5) - 0.3
    assert np.abs(np.hypot(ring, c[:, 2] - 0.5) - 0.1).mean() < 0.01        # jitter N(0, 0.005^2)
    c, n = inputs.make_cloud("bumpy", 20000)
    r = np.linalg.norm(c - 0.5, axis=1)
    assert r.min() >= 0.35 - 1e-6 and r.max() < 0.35 + 0.10   # overlapping bumps add
    # outward normals
    assert ((c - 0.5) * n).sum(1).min() > 0
    # occupancy like the paper's workloads: ~1-2.5 points per occupied cell at the config's resolution
    cfg, pts, _ = inputs.make_config(2)
    cells = np.unique((pts[0] * cfg.N).astype(np.int64) @ np.array([cfg.N * cfg.N, cfg.N, 1])).size
    assert 1.0 <= cfg.P / cells <= 2.5


WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_2106_03452_b200 import inputs
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# replica sharding of a batch: rank r owns items r, r+world, ... ; no data-path collective
cfg, pts, nrm = inputs.make_config(3, batch=4, P=500)
mine = list(range(rank, 4, world))
from oracle import dpsr_oracle as orc        # CPU stand-in for the per-rank solve in this host-logic test
local = torch.tensor([orc.forward(32, 2.0, pts[b], nrm[b])["mu"] for b in mine], dtype=torch.float64)
t = torch.tensor([1.0 + rank], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)     # the only cross-rank op: max-over-ranks timing
gathered = [torch.zeros_like(local) for _ in range(world)]
dist.all_gather(gathered, local)
if rank == 0:
    print(json.dumps({"max_t": t.item(), "mu": [g.tolist() for g in gathered], "items": [list(range(r, 4, world)) for r in range(world)]}))
dist.destroy_process_group()
"""


def test_world_size_2_replicas_gloo(tmp_path):
    import json
    from oracle import dpsr_oracle as orc
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29611", str(w), str(ROOT)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["max_t"] == 2.0 and d["items"] == [[0, 2], [1, 3]]
    cfg, pts, nrm = inputs.make_config(3, batch=4, P=500)
    for r, items in enumerate(d["items"]):
        for k, b in enumerate(items):
            assert abs(d["mu"][r][k] - orc.forward(32, 2.0, pts[b], nrm[b])["mu"]) < 1e-14
