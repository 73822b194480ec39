"""GPU tests of the coarse-to-fine driver (paper_2106_03452_b200/schedule.py): consecutive
{forward, backward, point update} iterations against the float64 oracle performing the same updates."""
import numpy as np
import pytest

from oracle import dpsr_oracle as orc
from paper_2106_03452_b200 import inputs

pytestmark = pytest.mark.gpu


def _oracle_update(N, pts, nrm, gp, gn, move=0.25):
    eta = move / N / max(np.abs(gp).max(), 1e-20)
    return np.clip(pts - eta * gp, 0.0, 1.0 - 1e-6), nrm - eta * gn


@pytest.mark.parametrize("path", ["throughput", "latency"])
def test_three_iterations_with_point_updates_at_64(path):
    import torch
    from paper_2106_03452_b200.schedule import CoarseToFine, Level
    N, P, sigma = 64, 5000, 2.0
    pts, nrm = inputs.make_cloud("torus", P, seed=21)
    G = inputs.upstream_grad(N, 1, seed=22)
    sched = CoarseToFine(P, levels=(Level(N, sigma, 3),), with_mesh=False, path=path)
    c, n = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda()
    tG = torch.from_numpy(G).cuda()
    op, on = pts.astype(np.float64), nrm.astype(np.float64)        # the oracle's own float64 trajectory
    for it in range(3):
        cur_p, cur_n = c.cpu().numpy()[0].copy(), n.cpu().numpy()[0].copy()
        b = sched.gradients(0, c, n, grad_chi=tG)
        torch.cuda.synchronize()
        # (1) this iteration against the oracle on the very points the GPU used (float32 bits)
        f = orc.forward(N, sigma, cur_p, cur_n)
        bk = orc.backward(N, sigma, cur_p, cur_n, f, G[0])
        assert np.abs(b["chi"].cpu().numpy()[0, ] - f["chi"]).max() <= 1e-4 * np.abs(f["chi"]).max(), it
        assert np.linalg.norm(b["gp"].cpu().numpy()[0] - bk["grad_points"]) <= 1e-3 * np.linalg.norm(bk["grad_points"]), it
        assert np.linalg.norm(b["gn"].cpu().numpy()[0] - bk["grad_normals"]) <= 1e-3 * np.linalg.norm(bk["grad_normals"]), it
        # (2) the update itself
        from paper_2106_03452_b200.schedule import sgd_update
        sgd_update(c, n, b["gp"], b["gn"], N)
        want_p, want_n = _oracle_update(N, cur_p.astype(np.float64), cur_n.astype(np.float64), bk["grad_points"], bk["grad_normals"])
        assert np.abs(c.cpu().numpy()[0] - want_p).max() <= 2e-6
        assert np.abs(n.cpu().numpy()[0] - want_n).max() <= 1e-5 * np.abs(want_n).max()
        # (3) the oracle's own trajectory, never re-synchronised with the GPU
        f2 = orc.forward(N, sigma, op, on)
        b2 = orc.backward(N, sigma, op, on, f2, G[0])
        op, on = _oracle_update(N, op, on, b2["grad_points"], b2["grad_normals"])
    assert np.abs(c.cpu().numpy()[0] - op).max() <= 1e-5          # three quarter-cell steps later the clouds still agree
    sched.close()


def test_run_level_eager_and_cuda_graph_agree():
    import torch
    from paper_2106_03452_b200.schedule import CoarseToFine, Level
    N, P = 32, 3000
    pts, nrm = inputs.make_cloud("sphere", P, seed=1)
    G = torch.from_numpy(inputs.upstream_grad(N, 1, seed=2)).cuda()
    outs = []
    for graph in (False, True):
        sched = CoarseToFine(P, levels=(Level(N, 2.0, 6),), with_mesh=False)
        c, n = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda()
        sched.run_level(0, c, n, grad_chi=G, cuda_graph=graph)
        torch.cuda.synchronize()
        outs.append(c.cpu().numpy())
        sched.close()
    assert np.abs(outs[0] - outs[1]).max() <= 1e-5


def test_full_loop_with_mesh_and_adam_moves_the_cloud_towards_the_target():
    # Sec.3.2 end to end on the device at 32^3: a sphere of source points is pulled towards a smaller target sphere; the
    # Chamfer loss between the extracted mesh and the target must go down
    import torch
    from paper_2106_03452_b200.schedule import CoarseToFine, Level
    N, P = 32, 3000
    src, nrm = inputs.sphere(P, seed=0, radius=0.3)
    tgt, _ = inputs.sphere(4000, seed=1, radius=0.22)
    sched = CoarseToFine(P, levels=(Level(N, 2.0, 40),), with_mesh=True, max_target_points=4000)
    c = torch.from_numpy(src[None].astype(np.float32)).cuda().requires_grad_(True)
    n = torch.from_numpy(nrm[None].astype(np.float32)).cuda().requires_grad_(True)
    t = torch.from_numpy(tgt.astype(np.float32)).cuda()
    with torch.no_grad():
        b = sched.gradients(0, c, n, target=t)
        torch.cuda.synchronize()
        first = b["loss"].item()
        V, T = b["counts"].cpu().tolist()
        assert V > 500 and T > 1000 and np.isfinite(first)
        opt = torch.optim.Adam([c, n], lr=2e-3)
        sched.run_level(0, c, n, target=t, optimizer=opt)
        b = sched.gradients(0, c, n, target=t)
        torch.cuda.synchronize()
        last = b["loss"].item()
    assert last < 0.7 * first, (first, last)
    sched.close()
