"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the float64 oracle,
element by element, on the same seeded inputs.  Bars (BASELINE.json north_star):
max|d chi| <= 1e-4 max|chi|; gradients <= 1e-3 relative L2."""
import numpy as np
import pytest

from oracle import dpsr_oracle as orc
from paper_2106_03452_b200 import inputs

pytestmark = pytest.mark.gpu

CHI_TOL = 1e-4
GRAD_TOL = 1e-3


def _gpu_run(N, sigma, pts, nrm, G, path="auto"):
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    B, P = pts.shape[0], pts.shape[1]
    h = Dpsr(N, sigma, B, P)
    h.set_path(path)
    tp, tn = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    chi = h.forward(tp, tn)
    stats = h.stats()
    out = dict(chi=chi.cpu().numpy(), stats=stats, fwd_launches=h.last_launch_count)
    if G is not None:
        gp, gn = h.backward(tp, tn, chi, torch.from_numpy(G).cuda())
        out.update(gp=gp.cpu().numpy(), gn=gn.cpu().numpy(), bwd_launches=h.last_launch_count)
    torch.cuda.synchronize()
    h.close()
    return out


def _check_item(N, sigma, pts, nrm, G, got_chi, got_stats, got_gp, got_gn):
    f = orc.forward(N, sigma, pts, nrm)
    err = np.abs(got_chi - f["chi"]).max() / np.abs(f["chi"]).max()
    assert err <= CHI_TOL, f"chi rel-max err {err:.3e}"
    assert abs(got_stats[0] - f["mu"]) <= 1e-4 * abs(f["a"])
    assert abs(got_stats[1] - f["a"]) <= 1e-4 * abs(f["a"])
    assert abs(got_stats[2] - f["s"]) <= 1e-4 * f["s"]
    if G is not None:
        b = orc.backward(N, sigma, pts, nrm, f, G)
        ep = np.linalg.norm(got_gp - b["grad_points"]) / np.linalg.norm(b["grad_points"])
        en = np.linalg.norm(got_gn - b["grad_normals"]) / np.linalg.norm(b["grad_normals"])
        assert ep <= GRAD_TOL and en <= GRAD_TOL, f"grad rel-L2 err points {ep:.3e} normals {en:.3e}"
    return err


# both implementations of the path (include/sap_dpsr.h, SAP_PATH_*): the 13-launch throughput path and the
# one-cooperative-kernel-per-direction latency path (N <= 128, batch * N <= #SMs)
PATHS = ["throughput", "latency"]


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("cfg_id", [1, 2])
def test_config_parity(cfg_id, path):
    cfg, pts, nrm = inputs.make_config(cfg_id)
    G = inputs.upstream_grad(cfg.N, 1)
    r = _gpu_run(cfg.N, cfg.sigma, pts, nrm, G, path)
    _check_item(cfg.N, cfg.sigma, pts[0], nrm[0], G[0], r["chi"][0], r["stats"][0], r["gp"][0], r["gn"][0])
    assert r["fwd_launches"] > 0 and r["bwd_launches"] > 0


@pytest.mark.parametrize("N,P,sigma,shape", [(64, 5000, 2.0, "torus"), (32, 777, 3.0, "ellipsoids3"),
                                             (64, 1, 0.0, "sphere"), (128, 4099, 5.0, "bumpy")])
@pytest.mark.parametrize("path", PATHS)
def test_other_sizes_and_ragged_point_counts(N, P, sigma, shape, path):
    pts, nrm = inputs.make_cloud(shape, P, seed=7)
    G = inputs.upstream_grad(N, 1, seed=3)
    r = _gpu_run(N, sigma, pts[None], nrm[None], G, path)
    _check_item(N, sigma, pts, nrm, G[0], r["chi"][0], r["stats"][0], r["gp"][0], r["gn"][0])


def test_batch_items_are_independent():
    # config 3 shape, small batch: item b of a batched call == the oracle on item b alone
    cfg, pts, nrm = inputs.make_config(3, batch=3, P=4000)
    G = inputs.upstream_grad(cfg.N, 3, seed=1)
    r = _gpu_run(cfg.N, cfg.sigma, pts, nrm, G)
    for b in range(3):
        _check_item(cfg.N, cfg.sigma, pts[b], nrm[b], G[b], r["chi"][b], r["stats"][b], r["gp"][b], r["gn"][b])


@pytest.mark.parametrize("path", PATHS)
def test_latency_path_small_batches(path):
    # several items per launch on the latency path (32^3: up to 4, 64^3: up to 2); item b == the oracle on item b alone
    for N, B, P in ((32, 4, 1500), (64, 2, 2500)):
        cfg, pts, nrm = inputs.make_config(3, batch=B, P=P)
        G = inputs.upstream_grad(N, B, seed=2)
        r = _gpu_run(N, 2.0, pts, nrm, G, path)
        for b in range(B):
            _check_item(N, 2.0, pts[b], nrm[b], G[b], r["chi"][b], r["stats"][b], r["gp"][b], r["gn"][b])


def test_paths_can_be_mixed_and_latency_needs_an_eligible_handle():
    import torch
    from paper_2106_03452_b200.binding import Dpsr, SapError
    N, P = 64, 3000
    pts, nrm = inputs.make_cloud("torus", P, seed=5)
    G = inputs.upstream_grad(N, 1, seed=6)
    f = orc.forward(N, 2.0, pts, nrm)
    b = orc.backward(N, 2.0, pts, nrm, f, G[0])
    h = Dpsr(N, 2.0, 1, P)
    assert h.path == "latency"            # SAP_PATH_AUTO at 64^3
    tp, tn, tG = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda(), torch.from_numpy(G).cuda()
    for fwd_path, bwd_path in (("latency", "throughput"), ("throughput", "latency")):
        h.set_path(fwd_path)
        chi = h.forward(tp, tn)
        h.set_path(bwd_path)
        gp, gn = h.backward(tp, tn, chi, tG)
        torch.cuda.synchronize()
        assert np.abs(chi.cpu().numpy()[0] - f["chi"]).max() <= CHI_TOL * np.abs(f["chi"]).max()
        assert np.linalg.norm(gp.cpu().numpy()[0] - b["grad_points"]) <= GRAD_TOL * np.linalg.norm(b["grad_points"])
        assert np.linalg.norm(gn.cpu().numpy()[0] - b["grad_normals"]) <= GRAD_TOL * np.linalg.norm(b["grad_normals"])
    assert len(h.fused_phases()) > 0
    h.close()
    big = Dpsr(128, 2.0, 2, 100)          # batch * N > #SMs: not eligible
    assert big.path == "throughput"
    with pytest.raises(SapError):
        big.set_path("latency")
    big.close()
    h128 = Dpsr(128, 2.0, 1, 100)          # eligible, but AUTO keeps the throughput path at 128^3
    assert h128.path == "throughput"
    h128.set_path("latency")
    assert h128.path == "latency"
    h128.close()


def test_splat_is_bit_reproducible_on_the_latency_path():
    # the latency path rasterises with integer (fixed-point) atomics: chi' is independent of the order of the adds;
    # only mu (double atomics over <= 148 partial sums) could differ in its last bits
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm = inputs.make_config(1)
    h = Dpsr(cfg.N, cfg.sigma, 1, cfg.P)
    h.set_path("latency")
    tp, tn = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    a = h.forward(tp, tn).clone()
    for _ in range(3):
        b = h.forward(tp, tn)
        assert (a - b).abs().max().item() <= 2e-7 * a.abs().max().item()
    h.close()


@pytest.mark.parametrize("path", PATHS)
def test_points_on_lattice_planes_and_wrap(path):
    # degenerate positions: exactly on vertices, in the last cell (periodic wrap), coincident pairs
    N, sigma = 32, 2.0
    pts, nrm = inputs.make_cloud("sphere", 500, seed=11)
    pts[:50] = np.round(pts[:50] * N) / N
    pts[50:60, 0] = (N - 0.25) / N
    pts[60:70, 2] = 0.0
    pts[70:80] = pts[80:90]
    nrm[70:80] = -nrm[80:90]
    r = _gpu_run(N, sigma, pts[None], nrm[None], None, path)
    _check_item(N, sigma, pts, nrm, None, r["chi"][0], r["stats"][0], None, None)


def _wrap_cloud(N, P, shape, seed, tile=32):
    """A cloud pushed against the faces of the cube: points in the first and last cell of every axis, points exactly
    on y-tile boundaries (multiples of tile/N: the bins of the N >= 256 kernels) and a few just below 1.0."""
    pts, nrm = inputs.make_cloud(shape, P, seed=seed)
    rng = np.random.default_rng(seed + 100)
    k = P // 10
    for a in range(3):
        pts[a * k:(a + 1) * k, a] = rng.uniform(0.0, 1.0 / N, k)                       # first cell
        pts[(3 + a) * k:(4 + a) * k, a] = rng.uniform(1.0 - 1.0 / N, 1.0 - 1e-7, k)    # last cell: +1 corner wraps to 0
    pts[6 * k:7 * k, 1] = (rng.integers(0, N // tile, k) * tile + rng.uniform(0.0, 1.0, k) * (rng.uniform(0, 1, k) < 0.5)) / N
    pts[7 * k:8 * k, 1] = (rng.integers(1, N // tile + 1, k) * tile - rng.uniform(0.0, 1.0, k)) / N
    pts = np.clip(pts, 0.0, np.float32(1.0 - 6e-8)).astype(np.float32)
    # gradients are undefined ON lattice planes: nudge coordinates that sit within 1e-3 cell of one
    t = pts.astype(np.float64) * N
    near = np.abs(t - np.round(t)) < 1e-3
    pts = np.where(near, (np.round(t) + 0.37) / N, pts).astype(np.float32)
    pts = np.clip(pts, 0.0, np.float32(1.0 - 6e-8)).astype(np.float32)
    return pts, nrm


def test_wrapping_points_forward_and_backward_batched_128():
    # periodic wrap through the backward (re-rasterised W, gather) with batch > 1
    N, P, B = 128, 3000, 2
    pts = np.empty((B, P, 3), np.float32)
    nrm = np.empty((B, P, 3), np.float32)
    for b in range(B):
        pts[b], nrm[b] = _wrap_cloud(N, P, "ellipsoids3", seed=20 + b)
    G = inputs.upstream_grad(N, B, seed=9)
    r = _gpu_run(N, 2.0, pts, nrm, G)
    for b in range(B):
        _check_item(N, 2.0, pts[b], nrm[b], G[b], r["chi"][b], r["stats"][b], r["gp"][b], r["gn"][b])


@pytest.mark.slow
def test_wrapping_points_forward_and_backward_256():
    # N >= 256 paths: y-tile wrap (ty + NTY - 1) % NTY, x-slab wrap with NTY > 1, transposed Nyquist planes
    N, P = 256, 20000
    pts, nrm = _wrap_cloud(N, P, "ellipsoids8", seed=31)
    G = inputs.upstream_grad(N, 1, seed=10)
    r = _gpu_run(N, 2.0, pts[None], nrm[None], G)
    _check_item(N, 2.0, pts, nrm, G[0], r["chi"][0], r["stats"][0], r["gp"][0], r["gn"][0])


@pytest.mark.parametrize("path", PATHS)
def test_non_unit_and_near_zero_normals(path):
    # normals are not normalised; a near-zero normal mutes its point
    N, P = 64, 4000
    pts, nrm = inputs.make_cloud("ellipsoids3", P, seed=12)
    rng = np.random.default_rng(5)
    nrm = (nrm * rng.uniform(0.2, 5.0, (P, 1))).astype(np.float32)
    nrm[:400] *= np.float32(1e-6)
    nrm[400:420] = 0.0
    G = inputs.upstream_grad(N, 1, seed=13)
    r = _gpu_run(N, 3.0, pts[None], nrm[None], G, path)
    _check_item(N, 3.0, pts, nrm, G[0], r["chi"][0], r["stats"][0], r["gp"][0], r["gn"][0])


@pytest.mark.parametrize("path", PATHS)
def test_backward_with_fewer_points_than_max_points(path):
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    N, Pmax, P = 64, 6000, 2500
    pts, nrm = inputs.make_cloud("torus", P, seed=14)
    G = inputs.upstream_grad(N, 1, seed=15)
    h = Dpsr(N, 2.0, 1, Pmax)
    h.set_path(path)
    tp, tn = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda()
    chi = h.forward(tp, tn)
    gp, gn = h.backward(tp, tn, chi, torch.from_numpy(G).cuda())
    torch.cuda.synchronize()
    _check_item(N, 2.0, pts, nrm, G[0], chi.cpu().numpy()[0], h.stats()[0], gp.cpu().numpy()[0], gn.cpu().numpy()[0])
    h.close()


def test_stale_forward_is_detected():
    # two forwards through one handle before a backward must not silently use the other cloud's state
    import torch
    from paper_2106_03452_b200.binding import Dpsr, SapError, dpsr
    N, P = 32, 1000
    h = Dpsr(N, 2.0, 1, P)
    clouds = [inputs.make_cloud(s, P, seed=3) for s in ("sphere", "torus")]
    tp = [torch.from_numpy(c[0][None].copy()).cuda().requires_grad_(True) for c in clouds]
    tn = [torch.from_numpy(c[1][None].copy()).cuda().requires_grad_(True) for c in clouds]
    f = dpsr(h)
    chi0 = f(tp[0], tn[0])
    e0 = h.epoch
    chi1 = f(tp[1], tn[1])                 # evaluation forward in between
    assert h.epoch == e0 + 1
    with pytest.raises(SapError):
        chi0.sum().backward()              # bins and statistics now belong to cloud 1
    chi1.sum().backward()                  # the latest forward is still differentiable
    assert tp[1].grad is not None
    # host forward followed by a device forward: backward_host must refuse
    hp, hn = torch.from_numpy(clouds[0][0][None].copy()), torch.from_numpy(clouds[0][1][None].copy())
    h.forward_host(hp, hn, None)
    h.forward(tp[1].detach(), tn[1].detach())
    with pytest.raises(SapError):
        h.backward_host(torch.zeros((1, N, N, N)), torch.empty((1, P, 3)), torch.empty((1, P, 3)))
    h.close()


def test_reserve_makes_first_fused_loss_call_capturable():
    # sap_dpsr_reserve: the optional buffers exist before the first call, so that call can be captured in a CUDA graph
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm = inputs.make_config(3, batch=1, P=2000)
    N = cfg.N
    h = Dpsr(N, cfg.sigma, 1, 2000)
    ws0 = h.workspace_bytes
    h.reserve(mse=True, host=True)
    assert h.workspace_bytes > ws0
    ws1 = h.workspace_bytes
    tp, tn = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    gt = torch.zeros((1, N, N, N), device="cuda")
    chi = torch.empty((1, N, N, N), device="cuda")
    loss = torch.empty((1,), device="cuda")
    gp, gn = torch.empty_like(tp), torch.empty_like(tn)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):          # very first forward_mse on this handle, inside capture
        h.forward_mse(tp, tn, gt, chi, loss)
        h.backward_mse(tp, tn, chi, gp, gn)
    graph.replay()
    torch.cuda.synchronize()
    assert h.workspace_bytes == ws1
    f = orc.forward(N, cfg.sigma, pts[0], nrm[0])
    assert abs(loss.item() - (f["chi"] ** 2).sum()) <= 1e-4 * (f["chi"] ** 2).sum()
    del graph
    h.close()


@pytest.mark.slow
def test_config4_256_parity_one_iteration():
    cfg, pts, nrm = inputs.make_config(4)
    G = inputs.upstream_grad(cfg.N, 1)
    r = _gpu_run(cfg.N, cfg.sigma, pts, nrm, G)
    _check_item(cfg.N, cfg.sigma, pts[0], nrm[0], G[0], r["chi"][0], r["stats"][0], r["gp"][0], r["gn"][0])


@pytest.mark.slow
def test_config3_full_batch32_parity():
    # BASELINE.json configs[2] at full size, the launch configuration bench.py times (batch 32 in one call)
    cfg, pts, nrm = inputs.make_config(3)
    G = inputs.upstream_grad(cfg.N, cfg.batch)
    r = _gpu_run(cfg.N, cfg.sigma, pts, nrm, G)
    for b in range(cfg.batch):
        _check_item(cfg.N, cfg.sigma, pts[b], nrm[b], G[b], r["chi"][b], r["stats"][b], r["gp"][b], r["gn"][b])


@pytest.mark.slow
def test_config5_512_parity():
    # BASELINE.json configs[4] at full size (512^3, 10^6 points), every voxel and every gradient against the naive
    # float64 oracle (about 3.5 minutes of 16 host cores)
    cfg, pts, nrm = inputs.make_config(5)
    G = inputs.upstream_grad(cfg.N, 1)
    r = _gpu_run(cfg.N, cfg.sigma, pts, nrm, G)
    _check_item(cfg.N, cfg.sigma, pts[0], nrm[0], G[0], r["chi"][0], r["stats"][0], r["gp"][0], r["gn"][0])


def test_fused_mse_loss_and_gradients():
    # learning-based setting (Eq.9): L = ||chi - chi_gt||^2 evaluated inside the normalisation pass
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm = inputs.make_config(3, batch=2, P=3000)
    N = cfg.N
    gt = (0.5 * np.tanh(inputs.upstream_grad(N, 2, seed=5))).astype(np.float32)   # some target grid in [-0.5, 0.5]
    h = Dpsr(N, cfg.sigma, 2, 3000)
    tp, tn = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    chi, loss = h.forward_mse(tp, tn, torch.from_numpy(gt).cuda())
    gp, gn = h.backward_mse(tp, tn, chi)
    # a plain forward/backward with the same G handed in from outside must agree with the fused path
    chi2 = h.forward(tp, tn)
    G = 2.0 * (chi2 - torch.from_numpy(gt).cuda())
    gp2, gn2 = h.backward(tp, tn, chi2, G)
    torch.cuda.synchronize()
    assert (gp - gp2).norm().item() <= 1e-4 * gp2.norm().item() and (gn - gn2).norm().item() <= 1e-4 * gn2.norm().item()
    for b in range(2):
        f = orc.forward(N, cfg.sigma, pts[b], nrm[b])
        d = f["chi"] - gt[b].astype(np.float64)
        assert abs(loss[b].item() - (d * d).sum()) <= 1e-4 * (d * d).sum()
        assert np.abs(chi[b].cpu().numpy() - f["chi"]).max() <= CHI_TOL * np.abs(f["chi"]).max()
        ref = orc.backward(N, cfg.sigma, pts[b], nrm[b], f, 2.0 * d)
        ep = np.linalg.norm(gp[b].cpu().numpy() - ref["grad_points"]) / np.linalg.norm(ref["grad_points"])
        en = np.linalg.norm(gn[b].cpu().numpy() - ref["grad_normals"]) / np.linalg.norm(ref["grad_normals"])
        assert ep <= GRAD_TOL and en <= GRAD_TOL, (ep, en)
    # the fused backward refuses to run after a plain forward
    from paper_2106_03452_b200.binding import SapError
    with pytest.raises(SapError):
        h.backward_mse(tp, tn, chi2)
    h.close()


def test_cuda_graph_replay_matches_eager():
    # forward and backward allocate nothing, never synchronise and keep no host-side state between calls, so a
    # captured CUDA graph (programmatic-dependent-launch edges included) can be replayed on new inputs
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    N, P = 64, 4000
    pts, nrm = inputs.make_cloud("torus", P, seed=2)
    pts2, nrm2 = inputs.make_cloud("ellipsoids3", P, seed=3)
    G = torch.from_numpy(inputs.upstream_grad(N, 1, seed=4)).cuda()
    h = Dpsr(N, 2.0, 1, P)
    c, n = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda()
    chi = torch.empty((1, N, N, N), dtype=torch.float32, device="cuda")
    gp, gn = torch.empty_like(c), torch.empty_like(n)

    def step():
        h.forward(c, n, chi)
        h.backward(c, n, chi, G, gp, gn)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        step()
    for p_, n_ in ((pts2, nrm2), (pts, nrm)):      # replay on other inputs written into the captured buffers
        c.copy_(torch.from_numpy(p_[None].copy()))
        n.copy_(torch.from_numpy(n_[None].copy()))
        graph.replay()
        torch.cuda.synchronize()
        got = (chi.clone(), gp.clone(), gn.clone())
        step()
        torch.cuda.synchronize()
        for a, b in zip(got, (chi, gp, gn)):
            assert (a - b).abs().max().item() <= 1e-5 * b.abs().max().item()
        f = orc.forward(N, 2.0, p_, n_)
        assert np.abs(got[0].cpu().numpy()[0] - f["chi"]).max() <= CHI_TOL * np.abs(f["chi"]).max()
    del graph
    h.close()


def test_repeatable_and_handle_reuse():
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm = inputs.make_config(1)
    h = Dpsr(cfg.N, cfg.sigma, 1, cfg.P)
    tp, tn = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    h.set_path("throughput")
    a = h.forward(tp, tn).clone()
    b = h.forward(tp, tn)
    # only the atomics' summation order may differ between two runs
    assert (a - b).abs().max().item() <= 1e-5 * a.abs().max().item()
    # fewer points than max_points on the same handle
    c = h.forward(tp[:, :1000].contiguous(), tn[:, :1000].contiguous())
    f = orc.forward(cfg.N, cfg.sigma, pts[0, :1000], nrm[0, :1000])
    assert np.abs(c.cpu().numpy()[0] - f["chi"]).max() <= CHI_TOL * np.abs(f["chi"]).max()
    h.close()


def test_host_buffer_entry_points_match_device_ones():
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm = inputs.make_config(1)
    G = inputs.upstream_grad(cfg.N, 1)
    r = _gpu_run(cfg.N, cfg.sigma, pts, nrm, G)
    h = Dpsr(cfg.N, cfg.sigma, 1, cfg.P)
    chi = torch.empty((1, cfg.N, cfg.N, cfg.N)).pin_memory()
    gp, gn = torch.empty((1, cfg.P, 3)).pin_memory(), torch.empty((1, cfg.P, 3)).pin_memory()
    h.forward_host(torch.from_numpy(pts), torch.from_numpy(nrm), chi)
    h.backward_host(torch.from_numpy(G), gp, gn)
    assert np.abs(chi.numpy() - r["chi"]).max() <= 1e-5 * np.abs(r["chi"]).max()
    assert np.linalg.norm(gp.numpy() - r["gp"]) <= 1e-4 * np.linalg.norm(r["gp"])
    assert np.linalg.norm(gn.numpy() - r["gn"]) <= 1e-4 * np.linalg.norm(r["gn"])
    h.close()


def test_autograd_function():
    import torch
    from paper_2106_03452_b200.binding import Dpsr, dpsr
    cfg, pts, nrm = inputs.make_config(1)
    G = inputs.upstream_grad(cfg.N, 1)
    h = Dpsr(cfg.N, cfg.sigma, 1, cfg.P)
    tp = torch.from_numpy(pts).cuda().requires_grad_(True)
    tn = torch.from_numpy(nrm).cuda().requires_grad_(True)
    chi = dpsr(h)(tp, tn)
    (chi * torch.from_numpy(G).cuda()).sum().backward()
    f = orc.forward(cfg.N, cfg.sigma, pts[0], nrm[0])
    b = orc.backward(cfg.N, cfg.sigma, pts[0], nrm[0], f, G[0])
    assert np.linalg.norm(tp.grad.cpu().numpy()[0] - b["grad_points"]) <= GRAD_TOL * np.linalg.norm(b["grad_points"])
    assert np.linalg.norm(tn.grad.cpu().numpy()[0] - b["grad_normals"]) <= GRAD_TOL * np.linalg.norm(b["grad_normals"])
    h.close()


# ---- activity lists ("nobody computes what nobody reads", sap_dpsr_set_sparse / sap_dpsr_get_activity) -----------------------
def _blob(P, centre, radius, seed):
    """points on a small sphere (a few active planes / tiles), periodic wrap when it sticks out of the cube"""
    rng = np.random.default_rng(seed)
    d = rng.normal(size=(P, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    pts = (np.asarray(centre)[None] + radius * d) % 1.0
    return pts.astype(np.float32), d.astype(np.float32)


def _active_counts(N, pts):
    """numpy restatement of the activity rule: tile (x, ty) is active when a point lies in bin (x | x-1, ty | ty-1)"""
    NL = N if N <= 128 else 32
    NTY = N // NL
    j = np.floor(pts.astype(np.float32) * np.float32(N)).astype(np.int64) % N
    cnt = np.zeros((N, NTY), np.int64)
    np.add.at(cnt, (j[:, 0], j[:, 1] // NL), 1)
    act = cnt + np.roll(cnt, 1, 0)
    if NTY > 1:
        act = act + np.roll(cnt, 1, 1) + np.roll(np.roll(cnt, 1, 0), 1, 1)
    ta = act > 0
    return int(ta.sum()), int(ta.any(1).sum())


def _run_sparse_dense(N, sigma, pts, nrm, G):
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    B, P = pts.shape[0], pts.shape[1]
    out = {}
    for mode in ("sparse", "dense"):
        h = Dpsr(N, sigma, B, P)
        h.set_path("throughput")
        h.set_sparse(mode == "sparse")
        tp, tn = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
        chi = h.forward(tp, tn)
        act = h.activity() if mode == "sparse" else None
        gp, gn = h.backward(tp, tn, chi, torch.from_numpy(G).cuda())
        torch.cuda.synchronize()
        out[mode] = dict(chi=chi.cpu().numpy(), gp=gp.cpu().numpy(), gn=gn.cpu().numpy(), act=act, stats=h.stats())
        if mode == "dense":
            with pytest.raises(Exception):
                h.activity()
        h.close()
    return out


@pytest.mark.parametrize("N,B,P", [(64, 2, 2500), (64, 10, 1500), (128, 3, 4000), (256, 1, 12000), (256, 2, 6000)])
def test_activity_lists_leave_results_unchanged(N, B, P):
    # items with very different activity: a small blob wrapping around the cube corner, a blob in the middle, a full-size shape
    # (batch 10 at 64^3: the throughput regime in which the solve masks the inactive planes instead of reading written zeros)
    pts = np.empty((B, P, 3), np.float32)
    nrm = np.empty((B, P, 3), np.float32)
    specs = [((0.02, 0.97, 0.5), 0.06), ((0.5, 0.52, 0.47), 0.11), None]
    for b in range(B):
        if specs[b % 3] is None:
            pts[b], nrm[b] = inputs.make_cloud("ellipsoids3", P, seed=40 + b)
        else:
            pts[b], nrm[b] = _blob(P, specs[b % 3][0], specs[b % 3][1], seed=40 + b)
    G = inputs.upstream_grad(N, B, seed=11)
    r = _run_sparse_dense(N, 2.0, pts, nrm, G)
    s, d = r["sparse"], r["dense"]
    # the skipped tiles hold zeros (forward) or values nobody reads (backward): same arithmetic on everything else (the
    # order of the points inside a bin, hence of the float sums of the point mean and the gather, varies from run to run)
    assert np.abs(s["chi"] - d["chi"]).max() <= 2e-6 * np.abs(d["chi"]).max()
    assert np.linalg.norm(s["gp"] - d["gp"]) <= 1e-5 * np.linalg.norm(d["gp"])
    assert np.linalg.norm(s["gn"] - d["gn"]) <= 1e-5 * np.linalg.norm(d["gn"])
    want_t = sum(_active_counts(N, pts[b])[0] for b in range(B))
    want_p = sum(_active_counts(N, pts[b])[1] for b in range(B))
    NTY = 1 if N <= 128 else N // 32
    assert s["act"] == (want_t, B * N * NTY, want_p, B * N)
    assert want_p < B * N    # the case does exercise skipped planes
    for b in range(B):
        _check_item(N, 2.0, pts[b], nrm[b], G[b], s["chi"][b], s["stats"][b], s["gp"][b], s["gn"][b])


@pytest.mark.parametrize("N,path", [(64, "latency"), (64, "throughput"), (128, "throughput"), (256, "throughput")])
def test_all_points_in_one_cell_and_a_volume_filling_cloud(N, path):
    # the two ends of the activity range, one item each in one batch:
    #  - 3000 points inside ONE cell with nearly parallel normals: every contribution lands on the same 8 nodes (the
    #    worst case of the shared-memory atomics and of the fixed-point scale, which is set from count x largest
    #    component), one or two active planes, every other plane / tile skipped by the listed kernels;
    #  - points uniform in the whole cube with random normals: every bin non-empty, every tile active (lists = dense)
    P, sigma = 3000, 2.0
    rng = np.random.default_rng(N)
    pts = np.empty((2, P, 3), np.float32)
    nrm = np.empty((2, P, 3), np.float32)
    cell = np.array([N // 2 + 3, N - 1, 17 % N], np.float64)        # the y index is the last cell: its +1 corner wraps
    pts[0] = ((cell[None] + rng.uniform(0.05, 0.95, (P, 3))) / N).astype(np.float32)
    d = np.array([0.3, -0.5, 0.81]) + 0.05 * rng.normal(size=(P, 3))
    nrm[0] = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    pts[1] = rng.uniform(0.0, 1.0, (P, 3)).astype(np.float32).clip(0.0, np.float32(1.0 - 6e-8))
    d = rng.normal(size=(P, 3))
    nrm[1] = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    G = inputs.upstream_grad(N, 2, seed=21)
    r = _gpu_run(N, sigma, pts, nrm, G, path)
    _check_item(N, sigma, pts[1], nrm[1], G[1], r["chi"][1], r["stats"][1], r["gp"][1], r["gn"][1])
    t0, p0 = _active_counts(N, pts[0])
    assert p0 == 2 and t0 <= 4                                       # one cell touches planes x and x + 1 only
    # Item 0 is the degenerate case of Eq.4 itself (reading R5 of DESIGN.md): a cloud inside one cell is a dipole, chi' is
    # antisymmetric about it, so its mean over the points m and chi'[0] are both ~1e-4 of max|chi'| and the scale
    # s = 0.5 / |chi'[0] - m| divides by their difference a.  An ABSOLUTE error eps max|chi'| of the float32 field (all
    # samples read the same 8 nodes: it does not average out) becomes a RELATIVE error eps kappa of s, kappa = max|chi'| / |a|,
    # in chi and in every gradient.  So: chi' and the statistics to the float32 bar, chi and the gradients to the bar times kappa.
    f = orc.forward(N, sigma, pts[0], nrm[0])
    chip_o = f["chi"] / f["s"] + f["mu"]
    M = np.abs(chip_o).max()
    kappa, eps = M / abs(f["a"]), 1e-6
    assert kappa > 500                                               # the case is what it claims to be (776 at 64^3, 4900 at 256^3)
    mu, a, sc = r["stats"][0][0], r["stats"][0][1], r["stats"][0][2]
    chip = r["chi"][0].astype(np.float64) / sc + mu
    assert np.abs(chip - chip_o).max() <= eps * M
    assert abs(mu - f["mu"]) <= eps * M and abs(a - f["a"]) <= eps * M
    bar = 2 * eps * kappa
    assert np.abs(r["chi"][0] - f["chi"]).max() <= max(CHI_TOL, bar) * np.abs(f["chi"]).max()
    bo = orc.backward(N, sigma, pts[0], nrm[0], f, G[0])
    for got, want in ((r["gp"][0], bo["grad_points"]), (r["gn"][0], bo["grad_normals"])):
        assert np.linalg.norm(got - want) <= max(GRAD_TOL, bar) * np.linalg.norm(want)


def test_single_launch_binning_matches_the_three_kernel_fallback(monkeypatch):
    # k_bin_sort (one cooperative launch) against k_bin_count / k_bin_scan / k_bin_scatter: same bins; the order of the
    # points inside a bin differs, which only reorders float sums in the point mean and nothing in the fixed-point splat
    N, P = 128, 7001
    pts, nrm = inputs.make_cloud("torus", P, seed=5)
    G = inputs.upstream_grad(N, 1, seed=12)
    a = _gpu_run(N, 2.0, pts[None], nrm[None], G, path="throughput")
    monkeypatch.setenv("SAP_BIN3", "1")
    b = _gpu_run(N, 2.0, pts[None], nrm[None], G, path="throughput")
    monkeypatch.delenv("SAP_BIN3")
    assert a["fwd_launches"] + 2 == b["fwd_launches"]
    assert np.abs(a["chi"] - b["chi"]).max() <= 2e-6 * np.abs(b["chi"]).max()
    assert np.linalg.norm(a["gp"] - b["gp"]) <= 1e-5 * np.linalg.norm(b["gp"])
    assert np.linalg.norm(a["gn"] - b["gn"]) <= 1e-5 * np.linalg.norm(b["gn"])
    _check_item(N, 2.0, pts, nrm, G[0], a["chi"][0], a["stats"][0], a["gp"][0], a["gn"][0])


def test_binning_with_several_points_per_thread_and_a_batch(monkeypatch):
    # from 65,536 points per item on k_bin_sort gives every thread four points (fewer blocks scan the counts and meet at the
    # grid barrier): two items of 70,000 points at 64^3, against the three-kernel binning and against the oracle
    N, P, B = 64, 70000, 2
    pts = np.empty((B, P, 3), np.float32)
    nrm = np.empty((B, P, 3), np.float32)
    pts[0], nrm[0] = inputs.make_cloud("torus", P, seed=61)
    pts[1], nrm[1] = inputs.make_cloud("ellipsoids3", P, seed=62)
    G = inputs.upstream_grad(N, B, seed=13)
    a = _gpu_run(N, 2.0, pts, nrm, G, path="throughput")
    monkeypatch.setenv("SAP_BIN3", "1")
    b = _gpu_run(N, 2.0, pts, nrm, G, path="throughput")
    monkeypatch.delenv("SAP_BIN3")
    assert a["fwd_launches"] + 2 == b["fwd_launches"]
    assert np.abs(a["chi"] - b["chi"]).max() <= 2e-6 * np.abs(b["chi"]).max()
    assert np.linalg.norm(a["gp"] - b["gp"]) <= 1e-5 * np.linalg.norm(b["gp"])
    assert np.linalg.norm(a["gn"] - b["gn"]) <= 1e-5 * np.linalg.norm(b["gn"])
    for i in range(B):
        _check_item(N, 2.0, pts[i], nrm[i], G[i], a["chi"][i], a["stats"][i], a["gp"][i], a["gn"][i])


def test_forward_on_one_path_backward_on_the_other_with_lists():
    # the latency path writes no activity lists: a throughput backward after it must fall back to every tile
    import torch
    from paper_2106_03452_b200.binding import Dpsr
    N, P = 64, 3000
    pts, nrm = _blob(P, (0.3, 0.3, 0.6), 0.12, seed=3)
    G = inputs.upstream_grad(N, 1, seed=13)
    h = Dpsr(N, 2.0, 1, P)
    tp, tn, tG = torch.from_numpy(pts[None]).cuda(), torch.from_numpy(nrm[None]).cuda(), torch.from_numpy(G).cuda()
    h.set_path("throughput")
    chi = h.forward(tp, tn)
    assert h.activity()[2] < N
    h.set_path("latency")
    chi = h.forward(tp, tn)
    with pytest.raises(Exception):
        h.activity()
    h.set_path("throughput")
    gp, gn = h.backward(tp, tn, chi, tG)
    torch.cuda.synchronize()
    _check_item(N, 2.0, pts, nrm, G[0], chi.cpu().numpy()[0], h.stats()[0], gp.cpu().numpy()[0], gn.cpu().numpy()[0])
    h.close()
