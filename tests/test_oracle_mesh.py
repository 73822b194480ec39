"""Pins of the mesh oracle (oracle/mesh_oracle.c): Marching Cubes, Eq.6 (L113-L117), Chamfer (L102).
Every check is against something other than the oracle itself: exactness on linear fields, topology of closed surfaces
(oriented 2-manifold, Euler characteristic), analytic radii / areas / volumes, hand-computed values, finite differences."""
import itertools

import numpy as np
import pytest

from oracle import mesh_oracle as mo


def _grid(N):
    g = np.arange(N) / N
    return np.meshgrid(g, g, g, indexing="ij")


def _directed_edges(tris):
    e = np.concatenate([tris[:, [0, 1]], tris[:, [1, 2]], tris[:, [2, 0]]])
    return e


def _is_closed_oriented_manifold(tris):
    """every directed edge appears exactly once and its reverse exactly once"""
    e = _directed_edges(tris)
    key = e[:, 0] * (tris.max() + 1) + e[:, 1]
    rkey = e[:, 1] * (tris.max() + 1) + e[:, 0]
    u, c = np.unique(key, return_counts=True)
    return bool((c == 1).all() and np.array_equal(np.sort(key), np.sort(rkey)))


def _euler(mesh):
    V = mesh["verts"].shape[0]
    F = mesh["tris"].shape[0]
    e = np.sort(_directed_edges(mesh["tris"]), axis=1)
    E = np.unique(e, axis=0).shape[0]
    return V - E + F


def _volume(mesh):
    p = mesh["verts"][mesh["tris"]]
    return np.einsum("ij,ij->i", p[:, 0], np.cross(p[:, 1], p[:, 2])).sum() / 6.0


def _area(mesh):
    p = mesh["verts"][mesh["tris"]]
    return 0.5 * np.linalg.norm(np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]), axis=1).sum()


def test_table_shape_and_trivial_cases():
    ntri, tris = mo.mc_table()
    assert ntri[0] == 0 and ntri[255] == 0
    assert ntri.max() <= mo.MC_MAX_TRI
    for c in range(8):                      # one corner inside: one triangle on the three edges at that corner
        assert ntri[1 << c] == 1 and ntri[255 ^ (1 << c)] == 1
    # a face of four inside corners (x = 0 face: corners 0, 2, 4, 6): a quad = 2 triangles on the four x edges (ids 0..3)
    cfg = (1 << 0) | (1 << 2) | (1 << 4) | (1 << 6)
    assert ntri[cfg] == 2 and set(tris[cfg, :2].ravel()) == {0, 1, 2, 3}
    # every crossed cube edge of a configuration is used, no other edge is
    for cfg in range(256):
        used = set(tris[cfg, :ntri[cfg]].ravel().tolist())
        crossed = set()
        for e in range(12):
            a, k = divmod(e, 4)
            others = [d for d in range(3) if d != a]
            o = [0, 0, 0]
            o[others[0]], o[others[1]] = k & 1, k >> 1
            c0 = o[0] | (o[1] << 1) | (o[2] << 2)
            c1 = c0 | (1 << a)
            if ((cfg >> c0) & 1) != ((cfg >> c1) & 1):
                crossed.add(e)
        assert used == crossed, cfg


def test_every_sign_configuration_gives_a_closed_oriented_surface():
    # each of the 256 configurations of one cube, embedded in an otherwise OUTSIDE 4^3 grid: the neighbouring cubes see
    # the shared faces with the same corner signs, so the surface must close (watertight across ambiguous faces)
    N = 4
    for cfg in range(1, 256):
        chi = np.ones((N, N, N))
        for c in range(8):
            if (cfg >> c) & 1:
                chi[1 + (c & 1), 1 + ((c >> 1) & 1), 1 + ((c >> 2) & 1)] = -1.0
        m = mo.marching_cubes(chi)
        assert m["tris"].shape[0] > 0
        assert _is_closed_oriented_manifold(m["tris"]), cfg
        assert _volume(m) > 0.0, cfg          # oriented outwards: the INSIDE region has positive volume


def test_random_sign_fields_close_away_from_the_boundary():
    rng = np.random.default_rng(0)
    N = 8
    chi = rng.standard_normal((N, N, N))
    chi[0], chi[-1], chi[:, 0], chi[:, -1], chi[:, :, 0], chi[:, :, -1] = (1.0,) * 6   # OUTSIDE shell: surface stays inside
    m = mo.marching_cubes(chi)
    assert _is_closed_oriented_manifold(m["tris"])


def test_linear_field_is_reproduced_exactly():
    N = 16
    X, Y, Z = _grid(N)
    chi = Z - (0.3017 + 0.2 * X + 0.1 * Y)         # plane z = 0.3017 + 0.2 x + 0.1 y, a graph over the whole cell box
    m = mo.marching_cubes(chi)
    p = m["verts"]
    assert np.abs(p[:, 2] - (0.3017 + 0.2 * p[:, 0] + 0.1 * p[:, 1])).max() < 1e-13
    side = (N - 1) / N
    assert abs(_area(m) - np.sqrt(1 + 0.2 ** 2 + 0.1 ** 2) * side ** 2) < 1e-12
    n = np.array([-0.2, -0.1, 1.0]) / np.sqrt(1 + 0.2 ** 2 + 0.1 ** 2)   # gradient direction of chi
    j = np.stack(np.unravel_index(m["vnode"], (N, N, N)), 1)
    interior = ((j >= 1) & (j <= N - 3)).all(1)   # central differences are exact away from the periodic wrap
    assert interior.sum() > 100
    assert np.abs(m["normals"][interior] - n).max() < 1e-12
    # geometric triangle normals point the same way (orientation: towards increasing chi)
    q = p[m["tris"]]
    fn = np.cross(q[:, 1] - q[:, 0], q[:, 2] - q[:, 0])
    assert (fn @ n > 0).all()


@pytest.mark.parametrize("N", [16, 32])
def test_sphere_topology_radius_volume_normals(N):
    X, Y, Z = _grid(N)
    c, r = np.array([0.47, 0.5, 0.52]), 0.31
    d = np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2)
    m = mo.marching_cubes(d - r)
    assert _is_closed_oriented_manifold(m["tris"])
    assert _euler(m) == 2
    rad = np.linalg.norm(m["verts"] - c, axis=1)
    h = 1.0 / N
    assert np.abs(rad - r).max() < h * h / r          # linear interpolation of a distance field: O(h^2) error
    assert abs(_volume(m) / (4 / 3 * np.pi * r ** 3) - 1) < 3 * h
    out = (m["verts"] - c) / rad[:, None]
    assert (np.einsum("ij,ij->i", m["normals"], out) > 0.98).all()
    assert np.abs(np.linalg.norm(m["normals"], axis=1) - 1).max() < 1e-12


def test_torus_has_genus_one():
    N = 32
    X, Y, Z = _grid(N)
    q = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2) - 0.28
    m = mo.marching_cubes(np.sqrt(q ** 2 + (Z - 0.5) ** 2) - 0.11)
    assert _is_closed_oriented_manifold(m["tris"]) and _euler(m) == 0


def test_two_spheres_two_components_and_exact_counts():
    N = 32
    X, Y, Z = _grid(N)
    d1 = np.sqrt((X - 0.3) ** 2 + (Y - 0.3) ** 2 + (Z - 0.3) ** 2) - 0.15
    d2 = np.sqrt((X - 0.7) ** 2 + (Y - 0.7) ** 2 + (Z - 0.7) ** 2) - 0.15
    m = mo.marching_cubes(np.minimum(d1, d2))
    assert _euler(m) == 4
    # vertex count == number of sign-changing grid edges, counted here with numpy
    ins = np.minimum(d1, d2) < 0
    V = (ins[1:] != ins[:-1]).sum() + (ins[:, 1:] != ins[:, :-1]).sum() + (ins[:, :, 1:] != ins[:, :, :-1]).sum()
    assert m["verts"].shape[0] == V


def test_dpsr_sphere_mesh_is_the_sphere():
    # the whole chain on config 1: oriented points on a sphere -> chi (DPSR oracle) -> mesh: a closed genus-0 surface
    # at the sphere's radius to within one cell (north_star / SURVEY 8(c))
    from oracle import dpsr_oracle as orc
    from paper_2106_03452_b200 import inputs
    cfg, pts, nrm = inputs.make_config(1)
    f = orc.forward(cfg.N, cfg.sigma, pts[0], nrm[0])
    m = mo.marching_cubes(f["chi"])
    assert _is_closed_oriented_manifold(m["tris"]) and _euler(m) == 2
    rad = np.linalg.norm(m["verts"] - 0.5, axis=1)
    assert np.abs(rad - 0.3).max() < 1.0 / cfg.N
    assert _volume(m) > 0 and (np.einsum("ij,ij->i", m["normals"], m["verts"] - 0.5) > 0).all()


def test_eq6_on_a_plane_by_hand():
    # plane x = c between node columns k and k+1: one vertex per (y, z) line at t = (c - k/N) N with normal +x.
    # dL/dp_v = (1, 0, 0) for every vertex  =>  g_v = -1, G[k, y, z] = -(1 - t), G[k+1, y, z] = -t, zero elsewhere.
    N, cpos = 8, 0.4
    X, _, _ = _grid(N)
    m = mo.marching_cubes(X - cpos)
    k = int(np.floor(cpos * N))
    t = cpos * N - k
    V = m["verts"].shape[0]
    assert V == N * N and np.allclose(m["vt"], t) and (m["vaxis"] == 0).all()
    dLdp = np.tile([1.0, 0.0, 0.0], (V, 1))
    G = mo.eq6_backward(N, m, dLdp)
    # interior lines only: the normal of a vertex next to the periodic wrap is not exactly +x
    assert np.allclose(G[k, 2:-2, 2:-2], -(1 - t)) and np.allclose(G[k + 1, 2:-2, 2:-2], -t)
    mask = np.ones(N, bool); mask[[k, k + 1]] = False
    assert np.abs(G[mask]).max() == 0.0
    # weights of a vertex sum to one: sum G = sum_v g_v
    rng = np.random.default_rng(1)
    d = rng.standard_normal((V, 3))
    assert abs(mo.eq6_backward(N, m, d).sum() + np.einsum("ij,ij->i", d, m["normals"]).sum()) < 1e-12


def test_chamfer_by_hand_and_properties():
    a = np.array([[0.0, 0, 0], [1, 0, 0]])
    b = np.array([[0.0, 0, 1]])
    r = mo.chamfer(a, b)
    assert r["nn_a"].tolist() == [0, 0] and r["nn_b"].tolist() == [0]
    assert np.allclose(r["dist_a"], [1, 2]) and np.allclose(r["dist_b"], [1])
    assert abs(r["loss"] - 2.5) < 1e-15
    # d/da0: (2/2)(a0 - b0) + (2/1)(a0 - b0) = 3 (0,0,-1); d/da1: (2/2)(a1 - b0) = (1,0,-1)
    assert np.allclose(r["grad_a"], [[0, 0, -3], [1, 0, -1]])
    rng = np.random.default_rng(2)
    p = rng.uniform(0, 1, (50, 3))
    assert mo.chamfer(p, p)["loss"] == 0.0
    q = rng.uniform(0, 1, (70, 3))
    assert abs(mo.chamfer(p, q)["loss"] - mo.chamfer(q, p)["loss"]) < 1e-15
    # against numpy's own distance matrix
    D = ((p[:, None, :] - q[None, :, :]) ** 2).sum(2)
    r = mo.chamfer(p, q)
    assert np.array_equal(r["nn_a"], D.argmin(1)) and np.array_equal(r["nn_b"], D.argmin(0))
    assert abs(r["loss"] - (D.min(1).mean() + D.min(0).mean())) < 1e-14


def test_chamfer_gradient_against_finite_differences():
    rng = np.random.default_rng(3)
    a, b = rng.uniform(0, 1, (12, 3)), rng.uniform(0, 1, (9, 3))
    r = mo.chamfer(a, b)
    h = 1e-6
    for i, d in itertools.product(range(12), range(3)):
        ap, am = a.copy(), a.copy()
        ap[i, d] += h; am[i, d] -= h
        fd = (mo.chamfer(ap, b, grads=False)["loss"] - mo.chamfer(am, b, grads=False)["loss"]) / (2 * h)
        assert abs(fd - r["grad_a"][i, d]) < 1e-7
    for k, d in itertools.product(range(9), range(3)):
        bp, bm = b.copy(), b.copy()
        bp[k, d] += h; bm[k, d] -= h
        fd = (mo.chamfer(a, bp, grads=False)["loss"] - mo.chamfer(a, bm, grads=False)["loss"]) / (2 * h)
        assert abs(fd - r["grad_b"][k, d]) < 1e-7
