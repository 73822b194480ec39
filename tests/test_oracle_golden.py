"""Regression guard: the oracle still produces the stored config-1 values (tests/golden/oracle_cfg1.txt,
written by tests/golden/make_golden.py from oracle/ only; Eq.2-4, Eq.5)."""
import os

import numpy as np

from oracle import dpsr_oracle as orc
from paper_2106_03452_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_cfg1.txt")


def load_golden():
    out = {"chi": {}, "grad_points": {}, "grad_normals": {}}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if t[0] in ("mu", "a", "s"):
            out[t[0]] = float(t[1])
        elif t[0] == "chi":
            out["chi"][tuple(int(x) for x in t[1:4])] = float(t[4])
        else:
            out[t[0]][int(t[1])] = np.array([float(x) for x in t[2:5]])
    return out


def test_oracle_reproduces_golden():
    g = load_golden()
    cfg, pts, nrm = inputs.make_config(1)
    f = orc.forward(cfg.N, cfg.sigma, pts[0], nrm[0])
    b = orc.backward(cfg.N, cfg.sigma, pts[0], nrm[0], f, inputs.upstream_grad(cfg.N)[0])
    for k in ("mu", "a", "s"):
        assert abs(f[k] - g[k]) <= 1e-11 * abs(g[k])
    for j, val in g["chi"].items():
        assert abs(f["chi"][j] - val) < 1e-11
    for i, val in g["grad_points"].items():
        assert np.abs(b["grad_points"][i] - val).max() < 1e-9
    for i, val in g["grad_normals"].items():
        assert np.abs(b["grad_normals"][i] - val).max() < 1e-10
