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

# Bytes a kernel must itself read once + write once ("compulsory"), in units of V = 4 N^3 per batch item: what
# roofline.achieved / roofline.frac are computed on (DESIGN.md 7 has the table).  The 52V per-axis-pass
# model of SURVEY 8(d) is a DIFFERENT quantity -- bytes an unfused one-pass-per-axis design would move -- and is only
# reported as `fusion_gain_vs_52V_model` (how many times fewer bytes than that model would need at the measured speed),
# never as a fraction of HBM peak.
YARD_FWD_BWD_V = 52.0
KERNEL_BYTES_V = {
    # label: (compulsory V for N <= 128 (y fused with z), compulsory V for N >= 256)
    "F:k_bin_sort": (0.0, 0.0), "F:k_bin_count": (0.0, 0.0), "F:k_bin_scan": (0.0, 0.0), "F:k_bin_scatter": (0.0, 0.0),   # 72 B/point, no grid traffic
    "F:k_zy_fwd": (3.0, 3.0),            # writes 3 spectra; the splatted field never exists in HBM
    "F:k_zw_fwd<SPLAT>": (3.0, 3.0),     # the same for N >= 256 (z pass only)
    "F:k_ring<FWD,y>": (0.0, 5.0),       # N >= 256 only: reads 3 spectra, writes 2 (x, u = h_y y + h_z z)
    "F:k_ring<SOLVE>": (4.0, 3.0),       # reads 3 (2) spectra, writes 1
    "F:k_ring<INV,y>": (0.0, 2.0),
    "F:k_zl_inv": (2.0, 2.0),            # reads 1 spectrum, writes chi'
    "F:k_zw_inv": (2.0, 2.0),            # the same for N >= 256 (z pass only)
    "F:k_sample_mean": (0.0, 0.0),       # gathers 8 values per point
    "F:k_scale_shift": (2.0, 2.0),
    "F:k_scale_shift_mse": (4.0, 4.0),
    "B:k_reduce_g": (2.0, 2.0),          # reads G and chi
    "B:k_zl_gbar": (2.0, 2.0),           # reads G, writes 1 spectrum (W is re-rasterised, not read)
    "B:k_zw_fwd<GBAR>": (2.0, 2.0),
    "B:k_ring<FWD,y>": (0.0, 2.0),
    "B:k_ring<ADJ>": (3.0, 3.0),         # reads 1 spectrum, writes 2 (x, B)
    "B:k_ring<INV,y>": (0.0, 5.0),       # reads 2 spectra, writes 3
    "B:k_zw_inv": (6.0, 6.0),            # N >= 256: reads 3 spectra, writes 3 grids
    "B:k_zl_inv": (5.0, 6.0),            # N <= 128: reads 2 spectra (B twice, the second time from L2), writes 3 grids
    "B:k_gather_grads": (0.0, 0.0),      # gathers 32 values per point
    # latency path: only chi (forward) / G and chi (backward) must cross HBM; the spectra live in L2 between the phases
    "F:k_fused_fwd": (1.0, 1.0), "B:k_fused_bwd": (2.0, 2.0),
}
# With the activity lists (sap_dpsr_get_activity: ft = active tiles / tiles, fp = active planes / planes) the listed kernels
# only move what a point can touch: their compulsory bytes scale with the fraction they process.
SPARSE_BYTES_V = {
    "F:k_zw_fwd<SPLAT>": lambda N, ft, fp: 3.0 * ft + 2.0 * (1.0 - fp),   # active tiles x 3 channels + the zeros of channels 0, 1 on inactive planes
    "F:k_ring<FWD,y>": lambda N, ft, fp: 5.0 * fp,             # 3 spectra in, 2 out, active planes only
    "B:k_ring<INV,y>": lambda N, ft, fp: 2.0 * fp + 3.0 * ft,  # 2 in on active planes, 3 out on active tiles
    "B:k_zl_inv": lambda N, ft, fp: (5.0 if N <= 128 else 6.0) * ft,   # active tiles only
    "B:k_zw_inv": lambda N, ft, fp: 6.0 * ft,
}


def compulsory_v(name, cfg, act):
    """bytes (in V) kernel `name` must read once + write once on this workload; act = (ft, fp) or None (dense)"""
    cv = KERNEL_BYTES_V.get(name, (0.0, 0.0))[0 if cfg.N <= 128 else 1]
    if act is not None and name in SPARSE_BYTES_V and cv > 0:
        cv = SPARSE_BYTES_V[name](cfg.N, act[0], act[1])
    if act is not None and name == "F:k_zy_fwd" and cfg.N <= 128 and cfg.batch * cfg.N >= 4 * 148:
        cv = 3.0 * act[0]   # throughput regime: the zeros of inactive planes are not written (the solve masks them)
    return cv


TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_traffic.json")


def load_traffic():
    """profiles/r02_traffic.json (written by paper_2106_03452_b200.profiling from an `ncu --set full` capture): per-launch
    dram bytes, valid only for the kernel sources it was captured at."""
    try:
        from paper_2106_03452_b200.profiling import kernel_tree_hash
        doc = json.load(open(TRAFFIC_JSON))
        if doc.get("kernel_sources") != kernel_tree_hash():
            return {}, f"stale (captured at kernel sources {doc.get('kernel_sources')}, running {kernel_tree_hash()})"
        return {k: v["bytes"] for k, v in doc["workloads"].items()}, f"profiles/r02_traffic.json @ {doc['kernel_sources']}"
    except Exception as e:   # no capture committed yet
        return {}, f"unavailable ({type(e).__name__})"


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


def time_config(cfg_id, steps, warmup, rank, torch, flush, with_e2e=True, with_profile=True, path="auto", custom=None):
    """Times `steps` forward+backward passes of BASELINE.json config cfg_id (or custom = (Config, pts, nrm, G)) on the
    current device: CUDA events on the launching stream, L2 flushed (256 MB write) before every step, outside the interval."""
    from paper_2106_03452_b200.binding import Dpsr
    cfg, pts, nrm, G = make_device_inputs(cfg_id, rank, torch) if custom is None else custom
    B, N, P = cfg.batch, cfg.N, cfg.P
    h = Dpsr(N, cfg.sigma, B, P)
    h.set_path(path)
    d_pts, d_nrm, d_G = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda(), torch.from_numpy(G).cuda()
    chi = torch.empty((B, N, N, N), dtype=torch.float32, device="cuda")
    gp, gn = torch.empty_like(d_pts), torch.empty_like(d_nrm)
    stream = torch.cuda.current_stream()

    launches = 0
    for _ in range(warmup):
        flush.zero_()
        h.forward(d_pts, d_nrm, chi, stream)
        h.backward(d_pts, d_nrm, chi, d_G, gp, gn, stream)
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
    act = None
    if h.path == "throughput":
        try:
            at, nt_, ap_, np_ = h.activity(stream)
            act = (at / max(nt_, 1), ap_ / max(np_, 1))
        except Exception:   # lists switched off
            act = None
    t_fwd = sum(a.elapsed_time(m) for a, m, b in ev)
    t_all = sum(a.elapsed_time(b) for a, m, b in ev)
    res = {"cfg": cfg, "ms_total": t_all, "ms_fwd": t_fwd / steps, "ms_bwd": (t_all - t_fwd) / steps,
           "ms_step": t_all / steps, "launches": launches, "workspace_bytes": h.workspace_bytes, "path": h.path,
           "activity": act}

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
        if h.path == "latency":
            res["fused_phases_us"] = dict(h.fused_phases())

    if with_e2e:       # host buffers through the C ABI: H2D points, normals, dL/dchi; D2H chi, gradients
        h.reserve(host=True)
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
    h.reserve(mse=True)
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


def _timed_loop(torch, fn, iters, warm=3):
    stream = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(iters):
        fn()
    b.record(stream)
    torch.cuda.synchronize()
    return a.elapsed_time(b) / iters


def _eager_and_graph(torch, it, iters):
    """ms per call of `it`, back to back from the host and replayed as a CUDA graph (the library allocates nothing and never
    synchronises, so an iteration can be captured)."""
    out = {"ms_per_iteration": _timed_loop(torch, it, iters)}
    try:
        stream = torch.cuda.current_stream()
        side = torch.cuda.Stream()
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            it()
        stream.wait_stream(side)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            it()
        out["ms_per_iteration_cuda_graph"] = _timed_loop(torch, graph.replay, iters)
        del graph
    except Exception as e:   # capture not supported in this environment: keep the eager number
        out["cuda_graph_error"] = str(e)[:200]
        torch.cuda.synchronize()
    return out


def time_config4_loop(torch, iters=100):
    """BASELINE.json configs[3] as stated: 100 CONSECUTIVE forward+backward iterations on the 100,000-point cloud at 256^3
    with a point update between them (points move by up to a quarter cell per iteration, so nothing about the binning can
    be cached).  Timed end to end with one pair of events around all iterations."""
    from paper_2106_03452_b200 import inputs
    from paper_2106_03452_b200.schedule import CoarseToFine, Level
    cfg, pts, nrm = inputs.make_config(4)
    sched = CoarseToFine(cfg.P, levels=(Level(cfg.N, cfg.sigma, iters),), with_mesh=False)
    c, n = torch.from_numpy(pts).cuda(), torch.from_numpy(nrm).cuda()
    G = torch.from_numpy(inputs.upstream_grad(cfg.N, 1)).cuda()

    def it():
        sched.run_level(0, c, n, iterations=1, grad_chi=G)
    out = _eager_and_graph(torch, it, iters)
    out["iterations"] = iters
    out["what"] = "forward + backward + point update per iteration, 100,000 points at 256^3, all iterations inside one timed interval (no L2 flush: consecutive iterations)"
    sched.close()
    return out


def time_coarse_to_fine(iters, torch):
    """The optimisation-based schedule of the paper (L121, L396) through paper_2106_03452_b200.schedule: 32^3 -> 64^3 ->
    128^3 (1000 iterations each, sigma 2, 2, 3) -> 256^3 (200 iterations, sigma 3) on 20,000 points.  Two legs per level:
    `dpsr` = forward + backward with a fixed upstream gradient + point update; `full` = the whole loop of Sec.3.2 on the
    device (DPSR forward, Marching Cubes, Chamfer to a 20,000-point target, Eq.6, DPSR backward, Adam step)."""
    from paper_2106_03452_b200 import inputs
    from paper_2106_03452_b200.schedule import CoarseToFine, paper_levels
    P = 20000
    pts, nrm = inputs.make_cloud("torus", P, seed=0)
    tgt, _ = inputs.make_cloud("ellipsoids3", P, seed=1)
    levels = paper_levels(3.0)
    out, total, total_full = {}, 0.0, 0.0
    for li, lv in enumerate(levels):
        entry = {"paper_iterations": lv.iterations, "sigma": lv.sigma}
        sched = CoarseToFine(P, levels=(lv,), with_mesh=True, max_target_points=P)
        c, n = torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda()
        G = torch.from_numpy(inputs.upstream_grad(lv.N, 1, seed=lv.N)).cuda()
        entry["path"] = sched.dpsr[0].path
        e = _eager_and_graph(torch, lambda: sched.run_level(0, c, n, iterations=1, grad_chi=G), iters)
        entry["dpsr"] = e
        total += min(v for k, v in e.items() if k.startswith("ms_")) * lv.iterations
        c2 = torch.from_numpy(pts[None].copy()).cuda().requires_grad_(True)
        n2 = torch.from_numpy(nrm[None].copy()).cuda().requires_grad_(True)
        t = torch.from_numpy(tgt).cuda()
        opt = torch.optim.Adam([c2, n2], lr=2e-3 * 0.7 ** li, capturable=True)
        with torch.no_grad():
            e = _eager_and_graph(torch, lambda: sched.run_level(0, c2, n2, iterations=1, target=t, optimizer=opt), iters)
            b = sched._buffers(0, c2.device)
            entry["full"] = dict(e, mesh_vertices=int(b["counts"][0].item()), mesh_triangles=int(b["counts"][1].item()),
                                 chamfer_loss=float(b["loss"].item()))
        total_full += min(v for k, v in e.items() if k.startswith("ms_")) * lv.iterations
        out[f"{lv.N}^3"] = entry
        sched.close()
    out["dpsr_ms_for_the_paper_schedule"] = total
    out["full_loop_ms_for_the_paper_schedule"] = total_full
    out["what"] = ("per level: ms per iteration on 20,000 points; totals = sum over levels of ms x the paper's iteration counts "
                   "(best of eager / CUDA graph; the eager full loop is bound by the host framework's optimiser step).  The paper's whole loop took 326-380 s per object on a 1080 Ti with "
                   "Marching Cubes on the CPU (Table 2, L166-L176)")
    return out


def time_cufft_comparison(cfg_ids, steps, torch, flush):
    """BENCH-ONLY yardstick (the product links no cuFFT): the library pipeline the paper describes (L84) for the
    same sizes -- torch.fft (cuFFT) 3 x rfftn + pointwise solve + 1 x irfftn forward, 1 x rfftn + pointwise + 3 x irfftn
    backward -- WITHOUT splat, normalisation or gather.  Same L2 flush and event protocol as the headline."""
    out = {}
    for cid in cfg_ids:
        from paper_2106_03452_b200 import inputs
        cfg = inputs.CONFIGS[cid]
        N, B = cfg.N, cfg.batch
        v = torch.randn((B, 3, N, N, N), device="cuda")
        g = torch.randn((B, N, N, N), device="cuda")
        k = torch.fft.fftfreq(N, 1.0 / N, device="cuda")
        kz = torch.fft.rfftfreq(N, 1.0 / N, device="cuda")
        KX, KY, KZ = torch.meshgrid(k, k, kz, indexing="ij")
        q = KX * KX + KY * KY + KZ * KZ
        f = torch.exp(-2.0 * cfg.sigma ** 2 * q / N ** 2) / (-2.0 * np.pi * q.clamp_min(1.0))
        f[0, 0, 0] = 0.0
        M = torch.stack([KX * f, KY * f, KZ * f]).to(torch.complex64) * 1j       # [3, N, N, N/2+1]

        def step():
            vh = torch.fft.rfftn(v, dim=(-3, -2, -1))
            chi = torch.fft.irfftn((vh * M).sum(1), s=(N, N, N), dim=(-3, -2, -1))
            gh = torch.fft.rfftn(g, dim=(-3, -2, -1))
            vb = torch.fft.irfftn(gh[:, None] * M.conj(), s=(N, N, N), dim=(-3, -2, -1))
            return chi, vb
        for _ in range(3):
            step()
        torch.cuda.synchronize()
        tot = 0.0
        for _ in range(steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            step()
            b.record()
            torch.cuda.synchronize()
            tot += a.elapsed_time(b)
        out[cfg.name] = {"ms_per_grid": tot / steps / B, "what": "cuFFT via torch.fft: 4 rfftn + 4 irfftn + 2 pointwise multiplies; no splat / normalise / gather"}
        del v, g, M, q, f, KX, KY, KZ
        torch.cuda.empty_cache()
    return out


def time_mesh_steps(torch, flush, N=128, P=20000, steps=10):
    """Marching Cubes / Chamfer / Eq.6 kernels alone (sap_mesh.h) on the indicator grid of a 20,000-point torus."""
    from paper_2106_03452_b200 import inputs
    from paper_2106_03452_b200.binding import Dpsr
    from paper_2106_03452_b200.mesh import Mesh
    pts, nrm = inputs.make_cloud("torus", P, seed=0)
    tgt, _ = inputs.make_cloud("torus", P, seed=1)
    d = Dpsr(N, 3.0, 1, P)
    m = Mesh(N, 12 * N * N, 24 * N * N, 12 * N * N)
    chi = d.forward(torch.from_numpy(pts[None].copy()).cuda(), torch.from_numpy(nrm[None].copy()).cuda())
    t = torch.from_numpy(tgt).cuda()
    verts, normals, tris, counts = m.extract(chi[0])
    loss, gv, _, _ = m.chamfer(verts, t, na_dev=counts)
    G = m.backward(gv, normals)
    torch.cuda.synchronize()
    out = {"N": N, "mesh_vertices": int(counts[0].item()), "mesh_triangles": int(counts[1].item()), "target_points": P}

    def timed(fn):
        tot = 0.0
        for _ in range(steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record()
            torch.cuda.synchronize()
            tot += a.elapsed_time(b)
        return tot / steps
    out["marching_cubes_ms"] = timed(lambda: m.extract(chi[0], verts, normals, tris, counts))
    out["chamfer_ms"] = timed(lambda: m.chamfer(verts, t, na_dev=counts, loss=loss, grad_a=gv))
    out["eq6_backward_ms"] = timed(lambda: m.backward(gv, normals, G))
    out["paper_context"] = "PAPER.md Table 4: Marching Cubes (CPU library) 0.039 s at 128^3, 0.374 s at 256^3"
    d.close(); m.close()
    return out


def roofline_of(res, peak_gbs, traffic):
    """Dominant kernel of the step (longest average launch) and its achieved bandwidth on the bytes the kernel itself must
    read once + write once (KERNEL_BYTES_V).  At 128^3 batch 1 the working set lives in the 126 MB L2, so the fraction says how
    far the launch is from streaming its compulsory bytes at HBM speed, not that it is HBM-bound."""
    cfg = res["cfg"]
    V = 4.0 * cfg.N ** 3 * cfg.batch
    km = res["kernels_ms"]
    name = max(km, key=km.get)
    comp_v = compulsory_v(name, cfg, res.get("activity"))
    ach = comp_v * V / (km[name] * 1e-3) / 1e9
    t = traffic.get(cfg.name, {}).get(name)
    return {"bound": "hbm", "kernel": name, "kernel_ms": km[name], "share_of_step": km[name] / sum(km.values()),
            "achieved": ach, "peak": peak_gbs, "unit": "GB/s", "frac": ach / peak_gbs, "traffic": t,
            "algorithmic_bytes": comp_v * V, "algorithmic_bytes_in_V": comp_v}


def kernel_fracs(res, peak_gbs):
    """compulsory bytes / time / measured peak for every grid kernel of the step"""
    cfg = res["cfg"]
    V = 4.0 * cfg.N ** 3 * cfg.batch
    out = {}
    for k, ms in res["kernels_ms"].items():
        cv = compulsory_v(k, cfg, res.get("activity"))
        if cv > 0:
            out[k] = round(cv * V / (ms * 1e-3) / 1e9 / peak_gbs, 3)
    return out


def activity_of(res):
    a = res.get("activity")
    if a is None:
        return None
    return {"active_tile_fraction": round(a[0], 4), "active_plane_fraction": round(a[1], 4),
            "what": "fraction of the 32-line tiles (planes for N <= 128) / x-planes a point can touch: the 3-channel y and z passes "
                    "process only those (sap_dpsr_get_activity); their compulsory bytes are scaled accordingly"}


def oracle_baseline(cfg_id, reps):
    """The float64 oracle as it stands on ONE grid of config cfg_id (512^3: a bounded sample, see `sample`)."""
    from oracle import dpsr_oracle as orc
    from paper_2106_03452_b200 import inputs
    cfg = inputs.CONFIGS[cfg_id]
    scale, N, P = 1.0, cfg.N, cfg.P
    if cfg.N > 256:    # 512^3 costs the oracle ~3.5 minutes: time the same shape at 256^3 with P/8 points, scale by the O(N^4) law
        N, P, scale = 256, cfg.P // 8, (cfg.N / 256.0) ** 4
    pts, nrm = inputs.make_cloud(cfg.shape, P, seed=0)
    G = inputs.upstream_grad(N, 1)[0]
    c = inputs.Config(cfg.name, N, 1, P, cfg.sigma, cfg.shape)
    t = min(oracle_step(c, pts, nrm, G) for _ in range(reps))
    sample = f"1 grid (N={N}, P={P}), forward+backward, best of {reps}"
    if scale != 1.0:
        sample += f"; x{scale:g} = (N_workload/N_sample)^4, the cost law of the oracle's naive separable DFT"
    return {"value": 1e3 * t * scale, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-based); default configs[1]")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="auto", choices=["auto", "throughput", "latency"], help="SAP_PATH_* of the headline handle")
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
    traffic, traffic_src = load_traffic()
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # headline: device-resident timing, barrier + synchronize on both sides, clocks sampled meanwhile
    barrier()
    with ClockSampler(local) as cs:
        res = time_config(args.config, args.steps, args.warmup, rank, torch, flush, with_e2e=False, with_profile=False, path=args.path)
        barrier()
    clocks = cs.summary()
    t_ms = torch.tensor([res["ms_total"]], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    t_total = float(t_ms.item())
    # per-kernel pass + end-to-end pass (separate so that their events/copies do not perturb `value`)
    res2 = time_config(args.config, args.steps, args.warmup, rank, torch, flush, with_e2e=True, with_profile=True, path=args.path)
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
                   "parallelism": f"replicas x{world} (no collective)", "l2": "flushed between steps (256 MB write)",
                   "path": res["path"]},
        "ms_fwd": res["ms_fwd"], "ms_bwd": res["ms_bwd"], "grids_per_s": 1e3 / value,
        "fusion_gain_vs_52V_model": {"what": "bytes the unfused per-axis-pass model of SURVEY 8(d) would move (52 V) / (time x measured HBM peak): "
                                             ">1 means the path is faster than that model could be at full HBM speed; NOT a fraction of peak",
                                     "value": YARD_FWD_BWD_V * V / (value * 1e-3) / 1e9 / (peak * world)},
        "clocks": clocks,
        "e2e": {"value": float(e2e.item()) / grids, "unit": UNIT, "h2d_bytes_per_step": res2["h2d"],
                "d2h_bytes_per_step": res2["d2h"]},
        "gpu_launches": res["launches"],
        "roofline": dict(roofline_of(res2, peak, traffic), peak_source=peak_src, traffic_source=traffic_src),
        "kernels_ms": res2["kernels_ms"],
        "kernel_frac_of_hbm_peak": kernel_fracs(res2, peak),
        "activity": activity_of(res2),
        "paper_context": "PAPER.md Table 4: 12 ms forward only at 128^3, 140 ms at 256^3, on a GTX 1080 Ti (not the target)",
    }
    solo = rank == 0 and world == 1
    if solo and args.also:
        also = {}
        for cid in [int(x) for x in args.also.split(",") if x.strip()]:
            if cid == args.config:
                continue
            k = max(3, min(args.steps, 20 if cid != 5 else 5))
            r = time_config(cid, k, 3, rank, torch, flush, with_e2e=False, with_profile=True)
            c = r["cfg"]
            Vc = 4.0 * c.N ** 3
            per_grid = r["ms_step"] / c.batch
            km = r["kernels_ms"]
            actual = sum(traffic.get(c.name, {}).values())
            also[c.name] = {"ms_per_grid": per_grid, "ms_fwd": r["ms_fwd"], "ms_bwd": r["ms_bwd"], "steps": k, "path": r["path"],
                            "grids_per_s": 1e3 / per_grid,
                            "fusion_gain_vs_52V_model": YARD_FWD_BWD_V * Vc / (per_grid * 1e-3) / 1e9 / peak,
                            "dram_bytes_per_fwd_bwd_in_V": (actual / (Vc * c.batch)) if actual else None,
                            "dram_GBps_actual": (actual / c.batch / (per_grid * 1e-3) / 1e9) if actual else None,
                            "roofline": roofline_of(r, peak, traffic), "kernels_ms": km,
                            "kernel_frac_of_hbm_peak": kernel_fracs(r, peak), "activity": activity_of(r)}
            if not args.no_cpu_baseline:
                also[c.name]["cpu_baseline"] = oracle_baseline(cid, 1)
        # both implementations of the path where the latency path applies
        from paper_2106_03452_b200 import inputs
        paths = {}
        for name, N, P, shape in (("32^3", 32, 3000, "sphere"), ("64^3", 64, 20000, "torus"), ("128^3", 128, 20000, "torus")):
            pts, nrm = inputs.make_cloud(shape, P, seed=0)
            custom = (inputs.Config(name, N, 1, P, 2.0, shape), pts[None].copy(), nrm[None].copy(), inputs.upstream_grad(N, 1))
            e = {}
            for path in ("throughput", "latency"):
                r = time_config(0, 20, 3, rank, torch, flush, with_e2e=False, with_profile=(path == "latency"), path=path, custom=custom)
                e[path + "_ms"] = r["ms_step"]
                if path == "latency":
                    e["latency_phases_us"] = r.get("fused_phases_us")
            paths[name] = e
        also["paths_throughput_vs_latency"] = paths
        if "4" in args.also.split(","):
            also["cfg4_100_iterations_with_point_updates"] = time_config4_loop(torch)
        also["cufft_comparison"] = time_cufft_comparison([c for c in (2, 3, 4, 5) if str(c) in args.also.split(",") or c == args.config], 5, torch, flush)
        also["coarse_to_fine_schedule"] = time_coarse_to_fine(20, torch)
        also["mesh_kernels_128"] = time_mesh_steps(torch, flush, 128)
        if "4" in args.also.split(","):
            also["mesh_kernels_256"] = time_mesh_steps(torch, flush, 256)
        if "3" in args.also.split(","):
            also["cfg3_fused_mse_loss"] = time_fused_mse(3, 10, 3, torch, flush)
        line["also"] = also
    if solo and not args.no_cpu_baseline:
        line["cpu_baseline"] = oracle_baseline(args.config, 3 if cfg.N <= 128 else 1)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
