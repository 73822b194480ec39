"""bench.py -- DPSR forward+backward on B200 (metric of BASELINE.json: ms per grid, fwd+bwd).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A step = one pass of the whole hot path (F1-F5 forward, B1-B6 backward) over one batch
of synthetic input.  Default workload: BASELINE.json configs[1] (128^3, batch 1, 20,000 torus points,
sigma 2).  `value` times the device-resident path with CUDA events (L2 flushed between steps, outside
the timed intervals); `e2e` times the host-buffer C-ABI calls (H2D/D2H inside).  Under torchrun each rank
runs the same workload on its own GPU (no collective in the data path: batch items are independent,
DESIGN.md "Multi-GPU"), the time is the max over ranks and the value the aggregate ("weak").
`--impl reference` times the float64 CPU oracle (oracle/) instead, as it stands.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "dpsr_fwd_bwd_ms_per_grid"
UNIT = "ms/grid"

# Algorithmic bytes per grid in units of V = 4 N^3 (SURVEY.md 8(d) per-axis-pass model): which table
# rows each of our kernels covers, and the bytes that kernel must itself read once + write once.
#   label: (yardstick V fused (N<=128), yardstick V unfused, compulsory V)   -- per channel-set launch
YARD_FWD_BWD_V = 52.0
KERNEL_BYTES_V = {
    # label: (yardstick V fused (N<=128), yardstick V unfused (N>=256), compulsory V fused, compulsory V unfused)
    # forward
    "F:k_bin_count": (0.0, 0.0, 0.0, 0.0),               # counting sort of the points (bytes ~ 72 B/point, ignored)
    "F:k_bin_scan": (0.0, 0.0, 0.0, 0.0),
    "F:k_bin_scatter": (0.0, 0.0, 0.0, 0.0),
    # splat fused in: rows "splat" (3V) + z r2c x3 (6V) [+ y x3 (6V) when fused]; it only WRITES 3V itself
    "F:k_zy_fwd": (15.0, 9.0, 3.0, 3.0),
    "F:k_ring<FWD,y>": (0.0, 6.0, 0.0, 5.0),             # row y sweep x3; writes 2 spectra (x, u = h_y y + h_z z)
    "F:k_ring<SOLVE>": (4.0, 4.0, 4.0, 3.0),             # row x sweep + solve + x inverse (3V or 2V in, 1V out)
    "F:k_ring<INV,y>": (0.0, 2.0, 0.0, 2.0),             # row inverse y
    "F:k_zl_inv": (4.0, 2.0, 2.0, 2.0),                  # rows [inverse y (2V) +] inverse z c2r (2V)
    "F:k_sample_mean": (0.0, 0.0, 0.0, 0.0),
    "F:k_scale_shift": (2.0, 2.0, 2.0, 2.0),             # row normalise
    # backward
    "B:k_reduce_g": (2.0, 2.0, 2.0, 2.0),                # row reductions
    "B:k_zl_gbar": (5.0, 3.0, 2.0, 2.0),                 # rows z r2c (G+W in, 1 out = 3V) + y (2V); W is re-rasterised, not read
    "B:k_zy_fwd<GBAR>": (5.0, 3.0, 2.0, 2.0),            # the same pass, one tile per CTA (N >= 256)
    "B:k_ring<FWD,y>": (0.0, 2.0, 0.0, 2.0),
    "B:k_ring<ADJ>": (4.0, 4.0, 4.0, 3.0),               # row x sweep + conj(M) fan-out + x inverses (1V in, 3V or 2V out)
    "B:k_ring<INV,y>": (0.0, 6.0, 0.0, 5.0),             # reads 2 spectra (x, B), writes 3
    "B:k_zl_inv": (12.0, 6.0, 6.0, 6.0),                 # rows inverse y x3 + inverse z x3
    "B:k_gather_grads": (4.0, 4.0, 0.0, 0.0),            # row gather (<= 4V, sparse)
}


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the `ncu --set full` captures summarised under
# profiles/r01_full_cfg{2,3,4}.md (one forward+backward each, kernels in launch order).  At 128^3 batch 1 the working
# set (~50 MB) lives in the 126 MB L2, so DRAM traffic is far BELOW the algorithmic bytes there.
NCU_TRAFFIC = {
    "cfg2_torus_128": {"F:k_bin_count": 244480, "F:k_bin_scan": 8704, "F:k_bin_scatter": 484864, "F:k_zy_fwd": 667648, "F:k_ring<SOLVE>": 25604096, "F:k_zl_inv": 8542976, "F:k_sample_mean": 2118400, "F:k_scale_shift": 8392192, "B:k_reduce_g": 16787968, "B:k_zl_gbar": 8739328, "B:k_ring<ADJ>": 8562944, "B:k_zl_inv": 25624832, "B:k_gather_grads": 7804160},
    "cfg3_ellipsoids_128_b32": {"F:k_zy_fwd": 773939712, "F:k_ring<SOLVE>": 1066452480, "F:k_zl_inv": 491010304, "F:k_scale_shift": 479487232, "B:k_reduce_g": 540808448, "B:k_zl_gbar": 495542528, "B:k_ring<ADJ>": 1032498688, "B:k_zl_inv": 1574035200},
    "cfg4_ellipsoids_256": {"F:k_zy_fwd": 147610880, "F:k_ring<FWD,y>": 284943616, "F:k_ring<SOLVE>": 166544896, "F:k_ring<INV,y>": 78128896, "F:k_zl_inv": 82979328, "F:k_scale_shift": 78618880, "B:k_reduce_g": 137347328, "B:k_zy_fwd<GBAR>": 92718336, "B:k_ring<FWD,y>": 78034432, "B:k_ring<ADJ>": 144984832, "B:k_ring<INV,y>": 280314112, "B:k_zl_inv": 350683648},
}


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clocks and throttle reasons while the timed region runs: NVML every 2 ms (the timed region of the
    128^3 workload is a few ms long), nvidia-smi every 100 ms if NVML cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None
        self.nvml, self.handle, self.max_mhz = None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        mhz = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
        r = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
        bits = [getattr(n, "nvmlClocksEventReasonHwSlowdown", 0x8), getattr(n, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                getattr(n, "nvmlClocksEventReasonSwThermalSlowdown", 0x20), getattr(n, "nvmlClocksEventReasonSwPowerCap", 0x4)]
        self.rows.append([mhz, self.max_mhz] + [bool(r & b) for b in bits])

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                             capture_output=True, text=True, timeout=5).stdout
        f = [x.strip() for x in out.strip().split(",")]
        if len(f) >= 6:
            self.rows.append([float(f[0]), float(f[1])] + [x.lower().startswith("active") for x in f[2:6]])

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample_nvml() if self.nvml else self._sample_smi()
            except Exception:
                pass
            self._stop.wait(0.002 if self.nvml else 0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(r[0] for r in self.rows)
        reasons = [n for i, n in enumerate(self.NAMES) if any(r[2 + i] for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.rows[0][1], "reasons": reasons, "samples": len(self.rows),
                "source": "nvml" if self.nvml else "nvidia-smi"}


def oracle_step(cfg, pts, nrm, G):
    """One forward+backward of the float64 oracle on ONE grid of the workload.  Returns seconds."""
    from oracle import dpsr_oracle as orc
    t0 = time.perf_counter()
    f = orc.forward(cfg.N, cfg.sigma, pts, nrm)
    orc.backward(cfg.N, cfg.sigma, pts, nrm, f, G)
    return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the same config / metric / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import dpsr_oracle as orc
    from paper_2106_03452_b200 import inputs
    cfg, pts, nrm = inputs.make_config(args.config, batch=1)
    G = inputs.upstream_grad(cfg.N, 1)[0]
    for _ in range(args.warmup):
        oracle_step(cfg, pts[0], nrm[0], G)
    ts = [oracle_step(cfg, pts[0], nrm[0], G) for _ in range(args.steps)]
    ms = 1e3 * float(np.sum(ts)) / args.steps
    cores = orc.num_threads()
    sample = f"1 grid of the workload per step (N={cfg.N}, P={cfg.P}), full forward+backward"
    line = {
        "impl": "reference", "metric": METRIC, "value": ms, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "N": cfg.N, "batch": 1, "points": cfg.P, "sigma": cfg.sigma},
        "cpu_baseline": {"value": ms, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": ms, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def make_device_inputs(cfg_id, rank, torch):
    from paper_2106_03452_b200 import inputs
    cfg, pts, nrm = inputs.make_config(cfg_id)
    G = inputs.upstream_grad(cfg.N, cfg.batch, seed=rank)
    return cfg, pts, nrm, G


def time_config(cfg_id, steps, warmup, rank, torch, flush, with_e2e=True, with_profile=True):
    """Times `steps` forward+backward passes of BASELINE.json config cfg_id on the current device."""
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm, G = make_device_inputs(cfg_id, rank, torch)
    B, N, P = cfg.batch, cfg.N, cfg.P
    h = Dpsr(N, cfg.sigma, B, P)
    d_pts, d_nrm, d_G = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda(), torch.from_numpy(G).cuda()
    chi = torch.empty((B, N, N, N), dtype=torch.float32, device="cuda")
    gp, gn = torch.empty_like(d_pts), torch.empty_like(d_nrm)
    stream = torch.cuda.current_stream()

    def step():
        h.forward(d_pts, d_nrm, chi, stream)
        nf = h.last_launch_count
        h.backward(d_pts, d_nrm, chi, d_G, gp, gn, stream)
        return nf + h.last_launch_count

    launches = 0
    for _ in range(warmup):
        flush.zero_()
        step()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(steps)]
    for a, m, b in ev:
        flush.zero_()          # L2 flush (buffer > 126 MB L2), outside the timed interval
        a.record(stream)
        h.forward(d_pts, d_nrm, chi, stream)
        launches += h.last_launch_count
        m.record(stream)
        h.backward(d_pts, d_nrm, chi, d_G, gp, gn, stream)
        launches += h.last_launch_count
        b.record(stream)
    torch.cuda.synchronize()
    t_fwd = sum(a.elapsed_time(m) for a, m, b in ev)
    t_all = sum(a.elapsed_time(b) for a, m, b in ev)
    res = {"cfg": cfg, "ms_total": t_all, "ms_fwd": t_fwd / steps, "ms_bwd": (t_all - t_fwd) / steps,
           "ms_step": t_all / steps, "launches": launches, "workspace_bytes": h.workspace_bytes}

    if with_profile:   # second pass with per-kernel events (their gaps would perturb the headline timing)
        h.set_profiling(True)
        acc = {}
        for _ in range(steps):
            flush.zero_()
            h.forward(d_pts, d_nrm, chi, stream)
            pf = h.profile()
            h.backward(d_pts, d_nrm, chi, d_G, gp, gn, stream)
            pb = h.profile()
            for name, ms in [("F:" + n, t) for n, t in pf] + [("B:" + n, t) for n, t in pb]:
                acc.setdefault(name, []).append(ms)
        h.set_profiling(False)
        res["kernels_ms"] = {k: float(np.mean(v)) for k, v in acc.items()}

    if with_e2e:       # host buffers through the C ABI: H2D points, normals, dL/dchi; D2H chi, gradients
        hp, hn, hG = (torch.from_numpy(x).pin_memory() for x in (pts, nrm, G))
        hchi = torch.empty((B, N, N, N), dtype=torch.float32).pin_memory()
        hgp, hgn = torch.empty((B, P, 3)).pin_memory(), torch.empty((B, P, 3)).pin_memory()
        for _ in range(min(warmup, 3)):
            h.forward_host(hp, hn, hchi, stream)
            h.backward_host(hG, hgp, hgn, stream)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            h.forward_host(hp, hn, hchi, stream)
            h.backward_host(hG, hgp, hgn, stream)
        torch.cuda.synchronize()
        res["e2e_ms_step"] = 1e3 * (time.perf_counter() - t0) / steps
        res["h2d"] = int(hp.numel() + hn.numel() + hG.numel()) * 4
        res["d2h"] = int(hchi.numel() + hgp.numel() + hgn.numel()) * 4
    h.close()
    del d_pts, d_nrm, d_G, chi, gp, gn
    torch.cuda.empty_cache()
    return res


def time_fused_mse(cfg_id, steps, warmup, torch, flush):
    """Learning-based setting (Eq.9): forward with the loss fused into the normalisation pass + backward from the
    gradient kept inside the handle (sap_dpsr_forward_mse / sap_dpsr_backward_mse); per grid, device-resident."""
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm, G = make_device_inputs(cfg_id, 0, torch)
    B, N, P = cfg.batch, cfg.N, cfg.P
    h = Dpsr(N, cfg.sigma, B, P)
    d_pts, d_nrm = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    d_gt = torch.from_numpy(np.tanh(G).astype(np.float32) * 0.5).cuda()
    chi = torch.empty((B, N, N, N), dtype=torch.float32, device="cuda")
    loss = torch.empty((B,), dtype=torch.float32, device="cuda")
    gp, gn = torch.empty_like(d_pts), torch.empty_like(d_nrm)
    stream = torch.cuda.current_stream()
    tot = 0.0
    for i in range(warmup + steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        h.forward_mse(d_pts, d_nrm, d_gt, chi, loss, stream)
        h.backward_mse(d_pts, d_nrm, chi, gp, gn, stream)
        b.record(stream)
        torch.cuda.synchronize()
        if i >= warmup:
            tot += a.elapsed_time(b)
    h.close()
    return {"ms_per_grid": tot / steps / B, "steps": steps, "what": "forward_mse + backward_mse (loss and dL/dchi never leave the handle)"}


def time_coarse_to_fine(iters, torch, flush):
    """The optimisation-based schedule of the paper (L121, L396): 32^3 -> 64^3 -> 128^3 (1000 iterations each, sigma
    2, 2, 3) -> 256^3 (200 iterations, sigma 3) on 20,000 points, one handle per level.  An iteration here = DPSR
    forward + backward + a gradient step on the points and normals (torch, on the device); Marching Cubes and the
    Chamfer loss of the paper's loop are out of scope, the upstream gradient is a fixed seeded grid.  `iters`
    iterations per level are timed and scaled to the paper's counts."""
    from paper_2106_03452_b200 import inputs
    from paper_2106_03452_b200.binding import Dpsr
    P = 20000
    pts, nrm = inputs.make_cloud("torus", P, seed=0)
    d_pts, d_nrm = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda()
    stream = torch.cuda.current_stream()
    out, total = {}, 0.0
    for N, sigma, n_it in ((32, 2.0, 1000), (64, 2.0, 1000), (128, 3.0, 1000), (256, 3.0, 200)):
        h = Dpsr(N, sigma, 1, P)
        G = torch.from_numpy(inputs.upstream_grad(N, 1, seed=N)).cuda()
        chi = torch.empty((1, N, N, N), dtype=torch.float32, device="cuda")
        gp, gn = torch.empty_like(d_pts), torch.empty_like(d_nrm)
        c, n = d_pts.clone(), d_nrm.clone()

        def it():
            h.forward(c, n, chi)
            h.backward(c, n, chi, G, gp, gn)
            step = 0.25 / N / gp.abs().max().clamp_min(1e-20)   # largest move: a quarter of a cell
            c.sub_(step * gp).clamp_(0.0, 1.0 - 1e-6)
            n.sub_(step * gn)

        def timed(fn):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(iters):
                fn()
            b.record(stream)
            torch.cuda.synchronize()
            return a.elapsed_time(b) / iters

        ms = timed(it)
        entry = {"ms_per_iteration": ms, "paper_iterations": n_it}
        try:   # the same iteration replayed as a CUDA graph: the library allocates nothing and never synchronises
            side = torch.cuda.Stream()
            side.wait_stream(stream)
            with torch.cuda.stream(side):
                it()
            stream.wait_stream(side)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                it()
            entry["ms_per_iteration_cuda_graph"] = timed(graph.replay)
            ms = min(ms, entry["ms_per_iteration_cuda_graph"])
            del graph
        except Exception as e:   # capture not supported in this environment: keep the eager number
            entry["cuda_graph_error"] = str(e)[:200]
            torch.cuda.synchronize()
        out[f"{N}^3"] = entry
        total += ms * n_it
        h.close()
    out["dpsr_ms_for_the_paper_schedule"] = total
    out["what"] = ("forward+backward+point update per iteration, 20,000 points; total = sum over levels of ms x the paper's "
                   "iteration counts (the paper's whole loop incl. Marching Cubes and Chamfer: 326-380 s per object on a 1080 Ti)")
    return out


def roofline_of(res, peak_gbs):
    """Dominant kernel of the step and its achieved bandwidth on the SURVEY 8(d) yardstick bytes."""
    cfg = res["cfg"]
    V = 4.0 * cfg.N ** 3 * cfg.batch
    fused = cfg.N <= 128
    km = res["kernels_ms"]
    name = max(km, key=km.get)
    yard_v, comp_v = (KERNEL_BYTES_V[name][0], KERNEL_BYTES_V[name][2]) if fused else (KERNEL_BYTES_V[name][1], KERNEL_BYTES_V[name][3])
    ach = yard_v * V / (km[name] * 1e-3) / 1e9
    comp = comp_v * V / (km[name] * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": name, "kernel_ms": km[name], "share_of_step": km[name] / sum(km.values()),
            "achieved": ach, "peak": peak_gbs, "unit": "GB/s", "frac": ach / peak_gbs,
            "traffic": NCU_TRAFFIC.get(cfg.name, {}).get(name),
            "algorithmic_bytes": yard_v * V, "achieved_compulsory": comp, "frac_compulsory": comp / peak_gbs,
            "compulsory_bytes": comp_v * V}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-based); default configs[1]")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--also", default="3,4,5", help="other configs to report under 'also' (rank 0, N=1 only); '' = none")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    if not torch.cuda.is_available():
        print(json.dumps({"error": "no CUDA device: the DPSR path has no CPU fallback"}))
        return 1
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peak, peak_src = read_peaks()
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # headline: device-resident timing, barrier + synchronize on both sides, clocks sampled meanwhile
    barrier()
    with ClockSampler(local) as cs:
        res = time_config(args.config, args.steps, args.warmup, rank, torch, flush, with_e2e=False, with_profile=False)
        barrier()
    clocks = cs.summary()
    t_ms = torch.tensor([res["ms_total"]], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    t_total = float(t_ms.item())
    # per-kernel pass + end-to-end pass (separate so that their events/copies do not perturb `value`)
    res2 = time_config(args.config, args.steps, args.warmup, rank, torch, flush, with_e2e=True, with_profile=True)
    e2e = torch.tensor([res2["e2e_ms_step"]], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(e2e, op=dist.ReduceOp.MAX)
    cfg = res["cfg"]
    grids = cfg.batch * world
    ms_step = t_total / args.steps
    value = ms_step / grids
    V = 4.0 * cfg.N ** 3
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": cfg.name, "N": cfg.N, "batch": cfg.batch, "points": cfg.P, "sigma": cfg.sigma,
                   "parallelism": f"replicas x{world} (no collective)", "l2": "flushed between steps (256 MB write)"},
        "ms_fwd": res["ms_fwd"], "ms_bwd": res["ms_bwd"], "grids_per_s": 1e3 / value,
        "path_GBps_52V": YARD_FWD_BWD_V * V / (value * 1e-3) / 1e9,
        "path_frac_52V": YARD_FWD_BWD_V * V / (value * 1e-3) / 1e9 / (peak * world),
        "clocks": clocks,
        "e2e": {"value": float(e2e.item()) / grids, "unit": UNIT, "h2d_bytes_per_step": res2["h2d"],
                "d2h_bytes_per_step": res2["d2h"]},
        "gpu_launches": res["launches"],
        "roofline": dict(roofline_of(res2, peak), peak_source=peak_src),
        "kernels_ms": res2["kernels_ms"],
        "paper_context": "PAPER.md Table 4: 12 ms forward only at 128^3, 140 ms at 256^3, on a GTX 1080 Ti (not the target)",
    }
    if rank == 0 and world == 1 and args.also:
        also = {}
        for cid in [int(x) for x in args.also.split(",") if x.strip()]:
            if cid == args.config:
                continue
            k = max(3, min(args.steps, 20 if cid != 5 else 5))
            r = time_config(cid, k, 3, rank, torch, flush, with_e2e=False, with_profile=True)
            c = r["cfg"]
            Vc = 4.0 * c.N ** 3
            per_grid = r["ms_step"] / c.batch
            also[c.name] = {"ms_per_grid": per_grid, "ms_fwd": r["ms_fwd"], "ms_bwd": r["ms_bwd"], "steps": k,
                            "grids_per_s": 1e3 / per_grid,
                            "path_frac_52V": YARD_FWD_BWD_V * Vc / (per_grid * 1e-3) / 1e9 / peak,
                            "roofline": roofline_of(r, peak), "kernels_ms": r["kernels_ms"]}
        line["also"] = also
    if rank == 0 and world == 1 and args.also:
        line["also"]["coarse_to_fine_schedule"] = time_coarse_to_fine(20, torch, flush)
    if rank == 0 and world == 1 and args.also and "3" in args.also.split(","):
        line["also"]["cfg3_fused_mse_loss"] = time_fused_mse(3, 10, 3, torch, flush)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import dpsr_oracle as orc
        from paper_2106_03452_b200 import inputs
        c, pts, nrm = inputs.make_config(args.config, batch=1)
        G = inputs.upstream_grad(c.N, 1)[0]
        reps = 3 if c.N <= 128 else 1
        t = min(oracle_step(c, pts[0], nrm[0], G) for _ in range(reps))
        line["cpu_baseline"] = {"value": 1e3 * t, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                                "sample": f"1 grid of the workload (N={c.N}, P={c.P}), forward+backward, best of {reps}"}
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
