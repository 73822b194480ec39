"""Coarse-to-fine driver of the optimisation-based setting (Sec.3.2; Suppl. B, L396): the source
point cloud is optimised at 32^3 -> 64^3 -> 128^3 (1000 iterations each) -> 256^3 (200 iterations) with
sigma = 2, 2, 3, {3 or 5}, learning rate 2e-3 decayed by 0.7 at every level, 20,000 source points.

One iteration, all on the device and without a host round trip (sizes of the mesh stay in device memory):
    chi = DPSR(points, normals)                     sap_dpsr_forward
    mesh = MarchingCubes(chi)                       sap_mc_extract        (L100)
    L, dL/dp_mesh = Chamfer(mesh vertices, target)  sap_chamfer           (L102)
    dL/dchi = Eq.6(dL/dp_mesh, n_mesh)              sap_mc_backward       (L113-L117)
    dL/dpoints, dL/dnormals                         sap_dpsr_backward     (Eq.5)
    optimiser step on points and normals            torch (Adam, L396) -- plumbing, not part of the hot path
This module only orchestrates handles (one Dpsr and one Mesh per level); every arithmetic step above runs in the
library's CUDA kernels.  Not done here (out of scope): the resampling of points from the largest mesh
component every 200 iterations (L119) -- the same points travel through all levels.

`fixed_grad` mode replaces the mesh part by a fixed upstream gradient dL/dchi (BASELINE.json configs[3]: "forward +
backward iterations with a point update between them"), with the plain update the bench and the tests use:
    eta = move / (N max|dL/dpoints|);  points <- clip(points - eta dL/dpoints, 0, 1);  normals <- normals - eta dL/dnormals
"""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class Level:
    N: int
    sigma: float
    iterations: int


def paper_levels(sigma_final: float = 3.0):
    """L121 / L396: sigma = 2 at 32^3 and 64^3, 3 at 128^3, 3 (detailed objects) or 5 (noisy inputs) at 256^3."""
    return (Level(32, 2.0, 1000), Level(64, 2.0, 1000), Level(128, 3.0, 1000), Level(256, float(sigma_final), 200))


_scratch = {}


def sgd_update(points, normals, gp, gn, N, move=0.25):
    """The plain update of the fixed-gradient mode, in place, on the device, no host sync (sap_points_sgd_step: two small
    kernels): eta = move / (N max|gp|); points <- clip(points - eta gp, 0, 1 - 1e-6); normals <- normals - eta gn."""
    import torch
    from .mesh import sgd_step
    key = points.device
    if key not in _scratch:
        _scratch[key] = torch.zeros((1,), dtype=torch.int32, device=points.device)
    sgd_step(points, normals, gp, gn, N, move, _scratch[key])


class CoarseToFine:
    """Handles for every level of a schedule, created once (nothing is allocated inside the loop)."""

    def __init__(self, num_points, levels=None, with_mesh=True, max_target_points=0, path="auto"):
        from .binding import Dpsr
        self.levels = tuple(paper_levels() if levels is None else levels)
        self.P = int(num_points)
        self.with_mesh = bool(with_mesh)
        self.dpsr, self.mesh, self._buf = [], [], []
        for lv in self.levels:
            d = Dpsr(lv.N, lv.sigma, 1, self.P)
            d.set_path(path)
            self.dpsr.append(d)
            if self.with_mesh:
                from .mesh import Mesh
                max_v, max_t = 12 * lv.N * lv.N, 24 * lv.N * lv.N      # a closed surface crosses O(N^2) grid edges
                self.mesh.append(Mesh(lv.N, max_v, max_t, max(max_v, int(max_target_points))))
            self._buf.append(None)

    def _buffers(self, li, device):
        import torch
        if self._buf[li] is None:
            lv = self.levels[li]
            b = dict(chi=torch.empty((1, lv.N, lv.N, lv.N), dtype=torch.float32, device=device),
                     gp=torch.empty((1, self.P, 3), dtype=torch.float32, device=device),
                     gn=torch.empty((1, self.P, 3), dtype=torch.float32, device=device))
            if self.with_mesh:
                m = self.mesh[li]
                b.update(verts=torch.empty((m.max_v, 3), dtype=torch.float32, device=device),
                         normals=torch.empty((m.max_v, 3), dtype=torch.float32, device=device),
                         tris=torch.empty((m.max_t, 3), dtype=torch.int32, device=device),
                         counts=torch.zeros((2,), dtype=torch.int32, device=device),
                         gv=torch.empty((m.max_v, 3), dtype=torch.float32, device=device),
                         G=torch.empty((lv.N, lv.N, lv.N), dtype=torch.float32, device=device),
                         loss=torch.zeros((1,), dtype=torch.float32, device=device))
            self._buf[li] = b
        return self._buf[li]

    def gradients(self, li, points, normals, target=None, grad_chi=None):
        """One forward + backward at level li.  Returns the buffer dict (chi, gp, gn, and with a mesh: verts, normals,
        tris, counts, loss, G).  Either `target` [K,3] (mesh mode) or `grad_chi` [1,N,N,N] (fixed-gradient mode)."""
        b = self._buffers(li, points.device)
        d = self.dpsr[li]
        d.forward(points, normals, b["chi"])
        if grad_chi is None:
            m = self.mesh[li]
            m.extract(b["chi"][0], b["verts"], b["normals"], b["tris"], b["counts"])
            m.chamfer(b["verts"], target, na_dev=b["counts"], loss=b["loss"], grad_a=b["gv"])
            m.backward(b["gv"], b["normals"], b["G"])
            grad_chi = b["G"][None]
        d.backward(points, normals, b["chi"], grad_chi, b["gp"], b["gn"])
        return b

    def run_level(self, li, points, normals, iterations=None, target=None, grad_chi=None, optimizer=None, move=0.25,
                  cuda_graph=False):
        """`iterations` iterations at level li, updating points / normals in place.  optimizer: a torch optimiser over
        [points, normals] (mesh mode; its .grad fields are filled here) or None for sgd_update.  With cuda_graph the
        iteration is captured once and replayed (the library allocates nothing and never synchronises)."""
        import torch
        lv = self.levels[li]
        n_it = lv.iterations if iterations is None else int(iterations)

        def it():
            b = self.gradients(li, points, normals, target, grad_chi)
            if optimizer is None:
                sgd_update(points, normals, b["gp"], b["gn"], lv.N, move)
            else:
                points.grad, normals.grad = b["gp"], b["gn"]
                optimizer.step()

        if not cuda_graph:
            for _ in range(n_it):
                it()
            return
        stream = torch.cuda.current_stream()
        side = torch.cuda.Stream()
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            it()                       # warm-up outside capture (first-use initialisation of torch kernels)
        stream.wait_stream(side)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):  # recorded, not executed
            it()
        for _ in range(max(n_it - 1, 0)):
            graph.replay()

    def run(self, points, normals, target=None, grad_chi_per_level=None, lr=2e-3, decay=0.7, iterations=None, cuda_graph=False):
        """The whole schedule (L121, L396).  Mesh mode: Adam on points and normals, learning rate lr * decay^level.
        Fixed-gradient mode: grad_chi_per_level[li] and the plain update.  Points and normals are updated in place."""
        import torch
        for li in range(len(self.levels)):
            if grad_chi_per_level is not None:
                self.run_level(li, points, normals, iterations, grad_chi=grad_chi_per_level[li], cuda_graph=cuda_graph)
            else:
                opt = torch.optim.Adam([points, normals], lr=lr * decay ** li, capturable=cuda_graph)
                self.run_level(li, points, normals, iterations, target=target, optimizer=opt, cuda_graph=cuda_graph)
        return points, normals

    def close(self):
        for h in self.dpsr + self.mesh:
            h.close()
        self.dpsr, self.mesh = [], []
