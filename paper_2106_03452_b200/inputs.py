"""Seeded synthetic inputs for the DPSR hot path (the five BASELINE.json configs).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests/bench.
It holds none of the method's arithmetic (no splat, FFT, solve, normalise): it only draws
oriented point clouds and upstream gradients.  Everything is generated on the host in float64
with numpy.random.default_rng(seed) and rounded once to float32, so the oracle (which promotes
those float32 values to double) and the GPU see the same bits.  Recipes: DESIGN.md "Inputs"
(stand-ins for the paper's ShapeNet / Thingi10K / SRB / D-FAUST clouds, PAPER.md:L53, L121,
L396, L419, which are not available here: closed surfaces in the unit cube, 1-2.5 points per
occupied cell).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    N: int
    batch: int
    P: int
    sigma: float
    shape: str


CONFIGS = {
    1: Config("cfg1_sphere_32", 32, 1, 3_000, 2.0, "sphere"),
    2: Config("cfg2_torus_128", 128, 1, 20_000, 2.0, "torus"),
    3: Config("cfg3_ellipsoids_128_b32", 128, 32, 15_000, 2.0, "ellipsoids3"),
    4: Config("cfg4_ellipsoids_256", 256, 1, 100_000, 2.0, "ellipsoids8"),
    5: Config("cfg5_bumpy_sphere_512", 512, 1, 1_000_000, 3.0, "bumpy"),
}


def _unit(rng, n):
    d = rng.standard_normal((n, 3))
    return d / np.linalg.norm(d, axis=1, keepdims=True)


def sphere(P, seed=0, radius=0.3):
    """Config 1: P points uniform on a sphere centred in the unit cube, exact outward unit normals."""
    rng = np.random.default_rng(seed)
    d = _unit(rng, P)
    return 0.5 + radius * d, d.copy()


def torus(P, seed=0, R=0.3, r=0.1, pos_noise=0.005, nrm_noise=0.05):
    """Config 2: area-uniform torus about the z axis; jittered positions, noisy renormalised normals."""
    rng = np.random.default_rng(seed)
    u = rng.uniform(0.0, 2.0 * np.pi, P)
    v = np.empty(P)
    filled = 0
    while filled < P:
        cand = rng.uniform(0.0, 2.0 * np.pi, 2 * (P - filled) + 16)
        keep = cand[rng.uniform(0.0, 1.0, cand.size) < (R + r * np.cos(cand)) / (R + r)]
        k = min(keep.size, P - filled)
        v[filled:filled + k] = keep[:k]
        filled += k
    ring = R + r * np.cos(v)
    c = np.stack([ring * np.cos(u), ring * np.sin(u), r * np.sin(v)], 1) + 0.5
    n = np.stack([np.cos(v) * np.cos(u), np.cos(v) * np.sin(u), np.sin(v)], 1)
    c = c + rng.normal(0.0, pos_noise, c.shape)
    n = n + rng.normal(0.0, nrm_noise, n.shape)
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    return c, n


def ellipsoid_union(P, n_ell, seed=0, nrm_noise=0.0):
    """Configs 3/4: surface of the union of n_ell random axis-aligned ellipsoids, area-weighted.

    Centres U[0.3,0.7]^3, semi-axes U[0.08,0.2].  A unit-sphere direction d on a uniformly chosen
    ellipsoid is accepted with probability (local area stretch)/(largest stretch of any ellipsoid),
    which makes the accepted set area-uniform over all ellipsoid surfaces; points strictly inside
    another ellipsoid are rejected.  Outward normals n ~ ((x-cx)/a^2, (y-cy)/b^2, (z-cz)/c^2).
    """
    rng = np.random.default_rng(seed)
    ctr = rng.uniform(0.3, 0.7, (n_ell, 3))
    ax = rng.uniform(0.08, 0.2, (n_ell, 3))
    smax = np.max(np.stack([ax[:, 1] * ax[:, 2], ax[:, 0] * ax[:, 2], ax[:, 0] * ax[:, 1]], 1))
    pts, nrm = [], []
    have = 0
    while have < P:
        m = 4 * (P - have) + 256
        e = rng.integers(0, n_ell, m)
        d = _unit(rng, m)
        a = ax[e]
        stretch = np.sqrt((a[:, 1] * a[:, 2] * d[:, 0]) ** 2 + (a[:, 0] * a[:, 2] * d[:, 1]) ** 2 +
                          (a[:, 0] * a[:, 1] * d[:, 2]) ** 2)
        ok = rng.uniform(0.0, 1.0, m) < stretch / smax
        x = ctr[e] + a * d
        for o in range(n_ell):
            inside = (((x - ctr[o]) / ax[o]) ** 2).sum(1) < 1.0 - 1e-9
            ok &= ~(inside & (e != o))
        x, e2 = x[ok], e[ok]
        g = (x - ctr[e2]) / ax[e2] ** 2
        g /= np.linalg.norm(g, axis=1, keepdims=True)
        pts.append(x)
        nrm.append(g)
        have += x.shape[0]
    c = np.concatenate(pts)[:P]
    n = np.concatenate(nrm)[:P]
    if nrm_noise > 0.0:
        n = n + rng.normal(0.0, nrm_noise, n.shape)
        n /= np.linalg.norm(n, axis=1, keepdims=True)
    return c, n


def bumpy_sphere(P, seed=0, radius=0.35, n_bumps=64, amp=0.02, width=0.05, chunk=65536):
    """Config 5: radial surface rho(d) = radius + sum_b amp exp(-|radius (d-d_b)|^2 / (2 width^2)),
    c = 0.5 + rho(d) d, analytic normals n ~ rho d - grad_tan rho."""
    rng = np.random.default_rng(seed)
    db = _unit(rng, n_bumps)
    d = _unit(rng, P)
    c = np.empty((P, 3))
    n = np.empty((P, 3))
    k = radius * radius / (width * width)
    for s in range(0, P, chunk):
        dd = d[s:s + chunk]
        diff = dd[:, None, :] - db[None, :, :]
        bump = amp * np.exp(-0.5 * k * (diff ** 2).sum(2))
        rho = radius + bump.sum(1)
        grad = -(bump[:, :, None] * (k * diff)).sum(1)
        grad_t = grad - (grad * dd).sum(1, keepdims=True) * dd
        nn = rho[:, None] * dd - grad_t
        n[s:s + chunk] = nn / np.linalg.norm(nn, axis=1, keepdims=True)
        c[s:s + chunk] = 0.5 + rho[:, None] * dd
    return c, n


def make_cloud(shape, P, seed=0):
    """float32 (points [P,3] in [0,1), normals [P,3]) for a named shape."""
    if shape == "sphere":
        c, n = sphere(P, seed)
    elif shape == "torus":
        c, n = torus(P, seed)
    elif shape == "ellipsoids3":
        c, n = ellipsoid_union(P, 3, seed)
    elif shape == "ellipsoids8":
        c, n = ellipsoid_union(P, 8, seed, nrm_noise=0.05)
    elif shape == "bumpy":
        c, n = bumpy_sphere(P, seed)
    else:
        raise ValueError(shape)
    c32 = np.ascontiguousarray(c, dtype=np.float32)
    n32 = np.ascontiguousarray(n, dtype=np.float32)
    assert c32.min() >= 0.0 and c32.max() < 1.0
    return c32, n32


def make_config(cfg_id, batch=None, P=None):
    """float32 (points [B,P,3], normals [B,P,3]) for BASELINE.json config cfg_id; item b uses seed b."""
    cfg = CONFIGS[cfg_id]
    B = cfg.batch if batch is None else batch
    P = cfg.P if P is None else P
    pts = np.empty((B, P, 3), np.float32)
    nrm = np.empty((B, P, 3), np.float32)
    for b in range(B):
        pts[b], nrm[b] = make_cloud(cfg.shape, P, seed=b)
    return cfg, pts, nrm


def upstream_grad(N, batch=1, seed=0):
    """G = dL/dchi ~ N(0,1) i.i.d. per voxel, float32 [B,N,N,N] (BASELINE.json configs)."""
    rng = np.random.default_rng(1_000_003 + seed)
    return rng.standard_normal((batch, N, N, N), dtype=np.float32)
