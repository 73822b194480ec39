"""Pins for the float64 oracle (oracle/dpsr_oracle.c): it is checked here against what the paper
and the mathematics fix, NOT against itself and never against the CUDA path.

Each test names the passage of /root/reference/PAPER.md (PAPER.md:Lnnn) it pins.  The paper prints no
worked numerical example, so the pins are closed forms, the O(N^6) definition, a library FFT (used
in tests only), brute force with a different formula, invariants and finite differences.
"""
import itertools

import numpy as np
import pytest

from oracle import dpsr_oracle as orc
from paper_2106_03452_b200 import inputs

RNG = np.random.default_rng(1234)


# ----------------------------------------------------------------------------- DFT (Eq.12/13, L356-L360)
def test_dft_matches_direct_triple_sum_8cubed():
    x = RNG.standard_normal((8, 8, 8)) + 1j * RNG.standard_normal((8, 8, 8))
    for sign in (-1, +1):
        sep = orc.dft3(x, sign)
        direct = orc.dft3(x, sign, direct=True)
        assert np.abs(sep - direct).max() < 1e-12 * np.abs(direct).max()


def test_direct_triple_sum_is_the_definition():
    # the O(N^6) routine itself against a hand-built exponential sum at a few k (python loops)
    N = 4
    x = RNG.standard_normal((N, N, N)) + 1j * RNG.standard_normal((N, N, N))
    out = orc.dft3(x, -1, direct=True)
    for k in [(0, 0, 0), (1, 2, 3), (3, 0, 1)]:
        s = 0j
        for j in itertools.product(range(N), repeat=3):
            s += x[j] * np.exp(-2j * np.pi * (k[0] * j[0] + k[1] * j[1] + k[2] * j[2]) / N)
        assert abs(out[k] - s) < 1e-12


@pytest.mark.parametrize("N", [6, 16, 32])
def test_dft_matches_library_fft(N):
    x = RNG.standard_normal((N, N, N)) + 1j * RNG.standard_normal((N, N, N))
    assert np.abs(orc.dft3(x, -1) - np.fft.fftn(x)).max() < 1e-11 * N ** 1.5
    assert np.abs(orc.dft3(x, +1) - np.fft.ifftn(x)).max() < 1e-13


def test_dft_axis_order_delta_and_parseval():
    N = 8
    # a delta at (1,2,3) must give exp(-2 pi i (kx + 2 ky + 3 kz)/N): catches transposed axes
    x = np.zeros((N, N, N))
    x[1, 2, 3] = 1.0
    k = np.arange(N)
    want = np.exp(-2j * np.pi * (k[:, None, None] * 1 + k[None, :, None] * 2 + k[None, None, :] * 3) / N)
    assert np.abs(orc.dft3(x, -1) - want).max() < 1e-13
    # constant <-> delta, inverse carries 1/N^3 (R8)
    ones = np.ones((N, N, N))
    f = orc.dft3(ones, -1)
    assert abs(f[0, 0, 0] - N ** 3) < 1e-9 and abs(np.abs(f).sum() - N ** 3) < 1e-9
    y = RNG.standard_normal((N, N, N))
    fy = orc.dft3(y, -1)
    assert abs((np.abs(fy) ** 2).sum() / N ** 3 - (y ** 2).sum()) < 1e-9  # Parseval
    assert np.abs(orc.dft3(fy, +1) - y).max() < 1e-13                     # round trip


# ----------------------------------------------------------------------------- splat (Eq.10-11)
def _hat_splat(N, pts, nrm):
    """Brute force with a different formula: vertex j receives n_i * prod_a hat(t_a - j_a) where
    hat is the periodic tent function max(0, 1 - |d|) -- the definition of trilinear weights."""
    v = np.zeros((3, N, N, N))
    W = np.zeros((N, N, N))
    for jx, jy, jz in itertools.product(range(N), repeat=3):
        for i in range(pts.shape[0]):
            w = 1.0
            for a, j in enumerate((jx, jy, jz)):
                d = (pts[i, a] * N - j + N / 2) % N - N / 2   # periodic signed distance in cells
                w *= max(0.0, 1.0 - abs(d))
            if w:
                v[:, jx, jy, jz] += w * nrm[i]
                W[jx, jy, jz] += w
    return v, W


@pytest.mark.parametrize("N", [4, 6])
def test_splat_brute_force_tent_functions(N):
    pts = RNG.uniform(0, 1, (25, 3))
    pts[0] = [0.99, 0.0, 0.51]       # wraps in x, on a vertex plane in y
    nrm = RNG.standard_normal((25, 3))
    v, W = orc.splat(N, pts, nrm)
    bv, bW = _hat_splat(N, pts, nrm)
    assert np.abs(v - bv).max() < 1e-13 and np.abs(W - bW).max() < 1e-13


def test_splat_invariants():
    N = 16
    pts = RNG.uniform(0, 1, (200, 3))
    nrm = RNG.standard_normal((200, 3))
    v, W = orc.splat(N, pts, nrm)
    # weights sum to one: sum_j v_j = sum_i n_i, sum_j W_j = P
    assert np.abs(v.sum(axis=(1, 2, 3)) - nrm.sum(0)).max() < 1e-11
    assert abs(W.sum() - 200) < 1e-11
    # linearity in the normals
    v2, _ = orc.splat(N, pts, 3.0 * nrm)
    assert np.abs(v2 - 3.0 * v).max() < 1e-12
    # a point exactly on a vertex deposits its normal there only
    p = np.array([[5 / N, 7 / N, 15 / N]])
    n = np.array([[1.0, -2.0, 3.0]])
    v1, W1 = orc.splat(N, p, n)
    assert np.allclose(v1[:, 5, 7, 15], n[0]) and abs(np.abs(v1).sum() - 6.0) < 1e-14
    assert W1[5, 7, 15] == 1.0
    # two coincident points with opposite normals cancel ("paired point clusters that self-cancel")
    pp = np.repeat(RNG.uniform(0, 1, (1, 3)), 2, 0)
    nn = np.array([[0.3, 0.4, -1.0], [-0.3, -0.4, 1.0]])
    v0, _ = orc.splat(N, pp, nn)
    assert np.abs(v0).max() == 0.0
    # z is the fastest axis: a point near (x=1/N, y=2/N, z=3.5/N) splits between z=3 and z=4
    vz, _ = orc.splat(N, np.array([[1 / N, 2 / N, 3.5 / N]]), np.array([[1.0, 0, 0]]))
    assert abs(vz[0, 1, 2, 3] - 0.5) < 1e-15 and abs(vz[0, 1, 2, 4] - 0.5) < 1e-15


def test_interp_reproduces_trilinear_functions():
    # trilinear interpolation is exact for f = a + b x + c y + d z + e xy ... away from the wrap
    N = 8
    j = np.arange(N) / N
    X, Y, Z = np.meshgrid(j, j, j, indexing="ij")
    f = 1.0 + 2 * X - 3 * Y + 0.5 * Z + 4 * X * Y * Z
    pts = RNG.uniform(0.0, (N - 1) / N - 1e-9, (50, 3))
    want = 1.0 + 2 * pts[:, 0] - 3 * pts[:, 1] + 0.5 * pts[:, 2] + 4 * pts[:, 0] * pts[:, 1] * pts[:, 2]
    assert np.abs(orc.interp(N, pts, f) - want).max() < 1e-13
    # and it is the transpose of the splat: <W-splat of unit weights, f> = sum_i interp(f, c_i)
    _, W = orc.splat(N, pts, np.zeros((50, 3)))
    assert abs((W * f).sum() - orc.interp(N, pts, f).sum()) < 1e-11


# ----------------------------------------------------------------------------- multiplier (Eq.3; Eq.14-16)
def test_multiplier_values_and_symmetries():
    N, sigma = 16, 2.0
    # hand-evaluated: k = (1,0,0): q=1, g=exp(-2*4/256), m_x = g/(-2 pi)
    m = orc.multiplier(N, sigma, 1, 0, 0)
    assert np.allclose(m, [np.exp(-8.0 / 256) / (-2 * np.pi), 0, 0], atol=1e-16)
    # negative frequency k = N-3 -> u = -3
    m = orc.multiplier(N, sigma, 0, N - 3, 2)
    q = 9 + 4
    g = np.exp(-2 * 4 * q / 256)
    assert np.allclose(m, [0, g * (-3) / (-2 * np.pi * q), g * 2 / (-2 * np.pi * q)], atol=1e-16)
    # DC is zero (R4); Nyquist derivative component is zero but |u|^2 keeps (N/2)^2 (R3)
    assert np.all(orc.multiplier(N, sigma, 0, 0, 0) == 0)
    m = orc.multiplier(N, sigma, N // 2, 1, 0)
    q = 64 + 1
    assert m[0] == 0 and abs(m[1] - np.exp(-8 * q / 256) / (-2 * np.pi * q)) < 1e-18
    # odd in k (so that the real field stays real and the adjoint is -M)
    for k in [(1, 2, 3), (5, 8, 15), (8, 8, 8), (0, 9, 4)]:
        mk = orc.multiplier(N, sigma, *k)
        mm = orc.multiplier(N, sigma, *[(-c) % N for c in k])
        assert np.allclose(mk, -mm, atol=0)
    # sigma = 0: no filter
    assert abs(orc.multiplier(N, 0.0, 2, 0, 0)[0] - 2 / (-2 * np.pi * 4)) < 1e-18


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("k0", [1, 3])
def test_plane_wave_closed_form(axis, k0):
    """v_axis(j) = sin(2 pi k0 j_axis/N), other channels 0  =>  Eq.3 gives
    chi'(j) = -exp(-2 sigma^2 k0^2/N^2) cos(2 pi k0 j_axis/N) / (2 pi k0).
    Pins the sign, the 2 pi factors, the literal Gaussian of Eq.3 (R6), which channel pairs with
    which axis, and that grad chi' = smoothed v (Eq.1)."""
    N, sigma = 16, 2.0
    j = np.arange(N)
    shape = [1, 1, 1]
    shape[axis] = N
    theta = (2 * np.pi * k0 * j / N).reshape(shape) * np.ones((N, N, N))
    v = np.zeros((3, N, N, N))
    v[axis] = np.sin(theta)
    vt = np.stack([orc.dft3(v[c], -1) for c in range(3)])
    cp = orc.dft3(orc.spectral_solve(N, sigma, vt), +1)
    want = -np.exp(-2 * sigma ** 2 * k0 ** 2 / N ** 2) * np.cos(theta) / (2 * np.pi * k0)
    assert np.abs(cp.imag).max() < 1e-15
    assert np.abs(cp.real - want).max() < 1e-14


def test_nyquist_wave_is_annihilated_and_output_real():
    # R3: the derivative multiplier vanishes at k = N/2, so v_x = (-1)^jx gives chi' = 0;
    # and for an arbitrary real field the inverse transform is real to rounding.
    N, sigma = 8, 2.0
    v = np.zeros((3, N, N, N))
    v[0] = ((-1.0) ** np.arange(N))[:, None, None]
    vt = np.stack([orc.dft3(v[c], -1) for c in range(3)])
    assert np.abs(orc.dft3(orc.spectral_solve(N, sigma, vt), +1)).max() < 1e-15
    v = RNG.standard_normal((3, N, N, N))
    vt = np.stack([orc.dft3(v[c], -1) for c in range(3)])
    cp = orc.dft3(orc.spectral_solve(N, sigma, vt), +1)
    assert np.abs(cp.imag).max() < 1e-15 * np.abs(cp.real).max() + 1e-17
    assert abs(cp.real.sum()) < 1e-12          # zero DC (R4)


def test_spectral_poisson_identity_with_library_fft():
    """Eq.1 in spectral form (Eq.14/15): -4 pi^2 |u|^2 FFT(chi') = 2 pi i (u . FFT(v)) g, checked with
    numpy's FFT on the oracle's v and chi' of a real point cloud (independent of the oracle's DFT)."""
    N, sigma = 16, 2.0
    pts, nrm = inputs.make_cloud("sphere", 500, seed=3)
    f = orc.forward(N, sigma, pts, nrm, intermediates=True)
    u1 = np.fft.fftfreq(N, 1.0 / N)
    U = np.stack(np.meshgrid(u1, u1, u1, indexing="ij"))
    q = (U ** 2).sum(0)
    Uh = U.copy()
    Uh[np.abs(U) == N / 2] = 0.0
    lhs = -4 * np.pi ** 2 * q * np.fft.fftn(f["chi_prime"])
    rhs = 2j * np.pi * (Uh * np.fft.fftn(f["v"], axes=(1, 2, 3))).sum(0) * np.exp(-2 * sigma ** 2 * q / N ** 2)
    assert np.abs(lhs - rhs).max() < 1e-10 * np.abs(rhs).max()
    assert f["imag_residue"] < 1e-12


def test_R3_equals_literal_full_spectrum_real_part():
    # DESIGN.md reading R3: zeroing the Nyquist derivative == applying Eq.3 literally with fftfreq
    # signs on the full complex spectrum and keeping the real part.
    N, sigma = 8, 2.0
    v = RNG.standard_normal((3, N, N, N))
    u1 = np.fft.fftfreq(N, 1.0 / N)
    U = np.stack(np.meshgrid(u1, u1, u1, indexing="ij"))
    q = (U ** 2).sum(0)
    q[0, 0, 0] = 1.0
    ct = np.exp(-2 * sigma ** 2 * q / N ** 2) * 1j * (U * np.fft.fftn(v, axes=(1, 2, 3))).sum(0) / (-2 * np.pi * q)
    ct[0, 0, 0] = 0
    lit = np.fft.ifftn(ct).real
    vt = np.stack([orc.dft3(v[c], -1) for c in range(3)])
    cp = orc.dft3(orc.spectral_solve(N, sigma, vt), +1).real
    assert np.abs(cp - lit).max() < 1e-15


# ----------------------------------------------------------------------------- normalisation (Eq.2/4, L79-L92)
def test_normalisation_constraints_and_scale_invariance():
    N, sigma = 16, 2.0
    pts, nrm = inputs.make_cloud("sphere", 800, seed=1)
    f = orc.forward(N, sigma, pts, nrm)
    chi = f["chi"]
    assert abs(abs(chi[0, 0, 0]) - 0.5) < 1e-14                      # abs(chi|x=0) = m (Eq.2)
    assert abs(orc.interp(N, pts, chi).mean()) < 1e-13               # mean of chi over the points = 0 (Eq.4)
    assert abs(abs(f["s"] * f["a"]) - 0.5) < 1e-14
    # chi = s (chi' - mu)
    assert np.abs(chi - f["s"] * (f["chi_prime"] - f["mu"])).max() < 1e-13
    # invariance under n -> alpha n, alpha > 0 (normals need not be unit)
    f2 = orc.forward(N, sigma, pts, 7.5 * nrm.astype(np.float64))
    assert np.abs(f2["chi"] - chi).max() < 1e-12
    # flipping all normals flips inside/outside but the corner stays |0.5|
    f3 = orc.forward(N, sigma, pts, -nrm.astype(np.float64))
    assert np.abs(f3["chi"] + chi).max() < 1e-12


def test_sphere_level_set_and_sign():
    """Outward normals on a sphere: zero level set at the radius within one cell, chi<0 inside,
    ~ +0.5 outside (R9; PAPER.md:L385 'valued +-0.5 inside and outside')."""
    cfg, pts, nrm = inputs.make_config(1)
    N = cfg.N
    f = orc.forward(N, cfg.sigma, pts[0], nrm[0])
    chi = f["chi"]
    assert chi[0, 0, 0] == pytest.approx(0.5, abs=1e-14)
    c = N // 2
    assert chi[c, c, c] < -0.4
    for line in (chi[c:, c, c], chi[c, c:, c], chi[c, c, c:]):
        i = int(np.argmax(line > 0))             # first positive sample walking outwards
        zero = (i - 1) + line[i - 1] / (line[i - 1] - line[i])
        assert abs(zero - 0.3 * N) < 1.0
    j = (np.arange(N) / N - 0.5)
    R = np.sqrt(j[:, None, None] ** 2 + j[None, :, None] ** 2 + j[None, None, :] ** 2)
    assert (chi[R < 0.3 - 2.0 / N] < 0).all() and (chi[R > 0.3 + 2.0 / N] > 0).all()
    assert abs(np.median(chi[R > 0.45]) - 0.5) < 0.05


# ----------------------------------------------------------------------------- whole forward vs library FFT
def test_forward_equals_numpy_restatement_small():
    # the five steps restated with numpy's FFT at N=8 (special case that reduces to library routines)
    N, sigma = 8, 3.0
    pts = RNG.uniform(0, 1, (60, 3))
    nrm = RNG.standard_normal((60, 3))
    f = orc.forward(N, sigma, pts, nrm, intermediates=True)
    vt = np.fft.fftn(f["v"], axes=(1, 2, 3))
    ct = np.zeros((N, N, N), complex)
    for k in itertools.product(range(N), repeat=3):
        ct[k] = 1j * (orc.multiplier(N, sigma, *k) * vt[(slice(None),) + k]).sum()
    cp = np.fft.ifftn(ct).real
    assert np.abs(cp - f["chi_prime"]).max() < 1e-15
    mu = orc.interp(N, pts, cp).mean()
    assert abs(mu - f["mu"]) < 1e-16


def test_chi_tilde_at_matches_grid_route():
    N, sigma = 16, 2.0
    pts, nrm = inputs.make_cloud("torus", 300, seed=5)
    f = orc.forward(N, sigma, pts, nrm)
    ct = np.fft.fftn(f["chi_prime"])
    for k in [(1, 0, 0), (3, 15, 7), (8, 2, 1), (0, 0, 5), (8, 8, 8)]:
        assert abs(orc.chi_tilde_at(N, sigma, pts, nrm, k) - ct[k]) < 1e-12 * np.abs(ct).max()


# ----------------------------------------------------------------------------- backward (Eq.5 third factor, L110)
def _loss(N, sigma, pts, nrm, G):
    return float((orc.forward(N, sigma, pts, nrm)["chi"] * G).sum())


def test_backward_matches_central_finite_differences():
    N, sigma, P = 8, 2.0, 40
    pts = RNG.uniform(0.05, 0.95, (P, 3))
    t = pts * N                                     # keep points >= 1e-3 cells away from lattice planes
    fr = t - np.floor(t)
    pts = (np.floor(t) + np.clip(fr, 1e-3, 1 - 1e-3)) / N
    nrm = RNG.standard_normal((P, 3))
    G = RNG.standard_normal((N, N, N))
    f = orc.forward(N, sigma, pts, nrm)
    b = orc.backward(N, sigma, pts, nrm, f, G)
    h = 1e-6
    fd_p = np.zeros((P, 3))
    fd_n = np.zeros((P, 3))
    for i in range(P):
        for a in range(3):
            for arr, fd in ((pts, fd_p), (nrm, fd_n)):
                old = arr[i, a]
                arr[i, a] = old + h
                lp = _loss(N, sigma, pts, nrm, G)
                arr[i, a] = old - h
                lm = _loss(N, sigma, pts, nrm, G)
                arr[i, a] = old
                fd[i, a] = (lp - lm) / (2 * h)
    assert np.linalg.norm(b["grad_points"] - fd_p) < 1e-6 * np.linalg.norm(fd_p)
    assert np.linalg.norm(b["grad_normals"] - fd_n) < 1e-6 * np.linalg.norm(fd_n)


def test_backward_invariants():
    N, sigma = 16, 2.0
    pts, nrm = inputs.make_cloud("sphere", 400, seed=2)
    G = RNG.standard_normal((N, N, N))
    f = orc.forward(N, sigma, pts, nrm)
    b = orc.backward(N, sigma, pts, nrm, f, G, intermediates=True)
    gbar = b["gbar"]
    scale = np.abs(gbar).sum()
    # shift and scale invariance of the normalisation: sum Gbar' = 0 and sum Gbar' chi' = 0
    assert abs(gbar.sum()) < 1e-12 * scale
    assert abs((gbar * f["chi_prime"]).sum()) < 1e-12 * scale * np.abs(f["chi_prime"]).max()
    # Euler homogeneity: chi is invariant to n -> alpha n, so sum_i n_i . dL/dn_i = 0
    gn = b["grad_normals"]
    assert abs((gn * nrm).sum()) < 1e-10 * np.linalg.norm(gn) * np.linalg.norm(nrm)


def test_adjoint_identity_of_the_spectral_operator():
    # <A v, w> = <v, A^T w> with A = IDFT . M . DFT (forward) and A^T = IDFT . conj(M) . DFT (backward)
    N, sigma = 8, 2.0
    v = RNG.standard_normal((3, N, N, N))
    w = RNG.standard_normal((N, N, N))
    vt = np.stack([orc.dft3(v[c], -1) for c in range(3)])
    Av = orc.dft3(orc.spectral_solve(N, sigma, vt), +1).real
    Atw_t = orc.spectral_adjoint(N, sigma, orc.dft3(w, -1))
    Atw = np.stack([orc.dft3(Atw_t[c], +1).real for c in range(3)])
    assert abs((Av * w).sum() - (v * Atw).sum()) < 1e-13 * np.abs(Av).max() * np.abs(w).sum()
