"""Writes tests/golden/oracle_cfg1.txt: values of the float64 ORACLE (oracle/ only -- never the CUDA
path) on BASELINE.json config 1 (32^3 sphere, 3,000 points, sigma=2, seed 0).

The paper (arXiv 2106.03452) prints no worked numerical example of chi, so this file is not a pin of
the oracle; it is a regression guard for it (a later change to the oracle's arithmetic must justify a
new golden file in its commit message) and a fixed target for the GPU parity tests.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import dpsr_oracle as orc  # noqa: E402
from paper_2106_03452_b200 import inputs  # noqa: E402

SAMPLES = [(0, 0, 0), (16, 16, 16), (16, 16, 25), (16, 16, 26), (3, 29, 11), (31, 31, 31), (10, 20, 30)]
POINTS = [0, 1, 1499, 2999]


def main():
    cfg, pts, nrm = inputs.make_config(1)
    G = inputs.upstream_grad(cfg.N)[0]
    f = orc.forward(cfg.N, cfg.sigma, pts[0], nrm[0])
    b = orc.backward(cfg.N, cfg.sigma, pts[0], nrm[0], f, G)
    lines = ["# oracle values, config 1 (N=32, P=3000, sigma=2, seed 0); written by tests/golden/make_golden.py",
             "# cites: Eq.2-4 PAPER.md:L79-L92 (forward), Eq.5 third factor L110 (backward)",
             f"mu {float(f['mu'])!r}", f"a {float(f['a'])!r}", f"s {float(f['s'])!r}"]
    for j in SAMPLES:
        lines.append(f"chi {j[0]} {j[1]} {j[2]} {float(f['chi'][j])!r}")
    for i in POINTS:
        gp, gn = b["grad_points"][i], b["grad_normals"][i]
        lines.append(f"grad_points {i} {float(gp[0])!r} {float(gp[1])!r} {float(gp[2])!r}")
        lines.append(f"grad_normals {i} {float(gn[0])!r} {float(gn[1])!r} {float(gn[2])!r}")
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_cfg1.txt")
    with open(out, "w") as fh:
        fh.write("\n".join(lines) + "\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
