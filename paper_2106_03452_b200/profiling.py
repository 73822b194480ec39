"""Turns ncu output into the committed text summaries under profiles/ and into profiles/<round>_traffic.json, the
per-launch DRAM traffic that bench.py reports as `roofline.traffic`.  Runs here (no GPU): it only reads files that a
`gpurun` call brought back (an `.ncu-rep` capture or the CSV of a `--metrics gpu__time_duration.sum` launch list) with
`ncu -i ... --page raw --csv`, and the library's SASS with `cuobjdump`.

    python -m paper_2106_03452_b200.profiling launches <launches.csv> <out.md> --cfg cfg2 --cmd "<full ncu command>"
    python -m paper_2106_03452_b200.profiling full <capture.ncu-rep> <out.md> --cfg cfg4 --cmd "<full ncu command>" \
           [--traffic-json profiles/r02_traffic.json]
    python -m paper_2106_03452_b200.profiling sass <out.md>

Every summary is stamped with the hash of the kernel sources it was taken at (kernel_tree_hash); bench.py prints
`traffic: null` when the stamp in the JSON is not the hash of the sources it runs.
"""
from __future__ import annotations

import argparse
import collections
import csv
import hashlib
import io
import json
import re
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}

# metric -> row label of the --set full summary table
FULL_METRICS = [
    ("gpu__time_duration.sum", "duration"), ("dram__bytes_read.sum", "dram read"), ("dram__bytes_write.sum", "dram write"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "dram % of ncu peak"), ("lts__t_bytes.sum", "L2 bytes"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "smem wavefronts"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smem bank conflicts"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared_op_atom.sum", "smem ATOMIC wavefronts"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_atom.sum", "smem ATOMIC bank conflicts"),
    ("l1tex__t_output_wavefronts_pipe_lsu_mem_global_op_atom.sum", "global atomic wavefronts"),
    ("sm__throughput.avg.pct_of_peak_sustained_elapsed", "SM throughput %"),
    ("sm__inst_issued.avg.pct_of_peak_sustained_active", "issue active %"),
    ("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "fma pipe %"),
    ("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "alu pipe %"),
    ("sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "lsu pipe %"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps active %"),
    ("launch__registers_per_thread", "regs/thread"), ("launch__shared_mem_per_block_dynamic", "dyn smem/block"),
    ("launch__waves_per_multiprocessor", "waves/SM"),
    ("smsp__average_warp_latency_issue_stalled_long_scoreboard.ratio", "stall long_scoreboard"),
    ("smsp__average_warp_latency_issue_stalled_short_scoreboard.ratio", "stall short_scoreboard"),
    ("smsp__average_warp_latency_issue_stalled_barrier.ratio", "stall barrier"),
    ("smsp__average_warp_latency_issue_stalled_mio_throttle.ratio", "stall mio_throttle"),
    ("smsp__average_warp_latency_issue_stalled_lg_throttle.ratio", "stall lg_throttle"),
    ("smsp__average_warp_latency_issue_stalled_math_pipe_throttle.ratio", "stall math_pipe"),
    ("smsp__average_warp_latency_issue_stalled_wait.ratio", "stall wait"),
    ("smsp__inst_executed.sum", "warp instructions"),
]


def kernel_tree_hash() -> str:
    """sha1 over the kernel sources and C headers of the library: the stamp of every profile."""
    h = hashlib.sha1()
    for p in sorted((PKG / "csrc").glob("*.cu*")) + sorted((ROOT / "include").glob("*.h")):
        h.update(p.name.encode())
        h.update(p.read_bytes())
    return h.hexdigest()[:12]


def short_name(n: str) -> str:
    n = n.replace("sap::", "").replace("sapm::", "").replace("void ", "")
    return n.split("(")[0]


RING_MODE = {"0": "FWD,y", "1": "INV,y", "2": "SOLVE", "3": "ADJ", "4": "FWD,y", "5": "INV,y"}


def bench_label(name: str, backward: bool) -> str:
    """Label used by bench.py's kernels_ms for an ncu kernel name (template arguments decoded)."""
    n = short_name(name)
    m = re.match(r"k_ring<(\d+), ?(\d+)>", n)
    pre = "B:" if backward else "F:"
    if m:
        return pre + f"k_ring<{RING_MODE[m.group(2)]}>"
    m = re.match(r"k_zy_fwd<(\d+), ?(\d+), ?(\w+), ?(\d+)", n)
    if m:
        return pre + ("k_zy_fwd<GBAR>" if m.group(4) == "1" else "k_zy_fwd")
    m = re.match(r"k_zw_fwd<(\d+), ?(\d+)>", n)
    if m:
        return pre + ("k_zw_fwd<GBAR>" if m.group(2) == "1" else "k_zw_fwd<SPLAT>")
    return pre + re.sub(r"<.*", "", n)


def _num(x: str) -> float:
    return float(x.replace(",", ""))


def summarise_launches(csv_path: str, cfg: str, cmd: str) -> str:
    rows = list(csv.reader(open(csv_path)))
    h = [i for i, r in enumerate(rows) if "Kernel Name" in r][0]
    hdr = rows[h]
    iK, iV, iG, iB = hdr.index("Kernel Name"), hdr.index("Metric Value"), hdr.index("Grid Size"), hdr.index("Block Size")
    d = collections.OrderedDict()
    for r in rows[h + 1:]:
        if len(r) <= iV:
            continue
        d.setdefault((short_name(r[iK])[:56], r[iG], r[iB]), []).append(_num(r[iV]) / 1e3)
    ours = {k: v for k, v in d.items() if k[0].startswith("k_")}
    tot = sum(sum(v) for v in ours.values())
    out = [f"# ncu launch list, {cfg}, kernel sources {kernel_tree_hash()}", "",
           "Command (under gpurun, directly after the same command exited 0 without ncu):", "", f"    {cmd}", "",
           "Per-launch times are cold-cache and serialised by the profiler: compare SHARES, not absolutes.  `share` is of the",
           f"time in this library's kernels (k_*); sum of their mean durations = {sum(sum(v) / len(v) for v in ours.values()):.1f} us.", "",
           "| kernel | launches | grid | block | mean us | share |", "|---|---|---|---|---|---|"]
    for k, v in d.items():
        share = f"{100 * sum(v) / tot:.1f}%" if k in ours else "(not ours: torch fill / copy)"
        out.append(f"| `{k[0]}` | {len(v)} | {k[1]} | {k[2]} | {sum(v) / len(v):.2f} | {share} |")
    return "\n".join(out) + "\n"


def read_full(rep: str):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    return rows[0], rows[1], rows[2:]


def summarise_full(rep: str, cfg: str, cmd: str):
    hdr, units, data = read_full(rep)
    col = {n: i for i, n in enumerate(hdr)}
    names = [short_name(r[col["Kernel Name"]]) for r in data]
    lines = [f"# ncu --set full summary, {cfg}, kernel sources {kernel_tree_hash()}", "",
             "Command (under gpurun, directly after the same command exited 0 without ncu):", "", f"    {cmd}", "",
             "Launches in capture order.  Times are under the profiler (replayed, cold): use them for ratios and counters, not as",
             "bench values.  `k_ring<N, MODE>`: MODE 0 = FWD(y), 1 = INV(y), 2 = SOLVE, 3 = ADJ, 4 = FWD3, 5 = INV3; `k_zy_fwd<N, NL, FUSED_Y,",
             "SRC, NT>` and `k_zw_fwd<N, SRC>`: SRC 0 = SPLAT, 1 = GBAR.  `dram % of ncu peak` is of ncu's own peak (about 8.2 TB/s); the measured copy bandwidth",
             "(MEASURED_PEAKS.json, 6.54 TB/s) is 80 % of it.  `dram read` + `dram write` per launch is `roofline.traffic` in bench.py.", "",
             "| metric | " + " | ".join(f"`{n}`" for n in names) + " |", "|---|" + "---|" * len(names),
             "| grid | " + " | ".join(r[col["Grid Size"]] for r in data) + " |"]

    def fmt(x):
        try:
            return f"{_num(x):.4g}"
        except ValueError:
            return x
    for m, lab in FULL_METRICS:
        if m in col:
            lines.append(f"| {lab} [{units[col[m]]}] | " + " | ".join(fmt(r[col[m]]) for r in data) + " |")
    traffic = []
    for r in data:
        by = 0.0
        for m in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            by += _num(r[col[m]]) * UNIT[units[col[m]]]
        traffic.append((r[col["Kernel Name"]], int(by)))
    return "\n".join(lines) + "\n", traffic


def traffic_by_label(traffic):
    """One forward+backward in launch order -> {bench label: bytes}; the backward starts at k_reduce_g / k_fused_bwd."""
    out, backward = {}, False
    for name, by in traffic:
        n = short_name(name)
        if n.startswith("k_reduce_g") or n.startswith("k_fused_bwd"):
            backward = True
        lab = bench_label(name, backward)
        if lab not in out:          # first occurrence = one forward+backward
            out[lab] = by
    return out


SASS_OPS = ["UTMALDG", "UBLKCP", "SYNCS", "FFMA2", "FADD2", "FMUL2", "FFMA", "ATOMS", "ATOMG", "REDG", "RED", "BAR", "LDS", "STS",
            "LDG", "STG", "SHFL", "ACQBULK", "MATCH", "CCTL"]


def summarise_sass() -> str:
    lib = PKG / "libsap_dpsr.so"
    sass = subprocess.run(["cuobjdump", "-sass", str(lib)], capture_output=True, text=True, check=True).stdout
    per, cur = collections.OrderedDict(), None
    arch = sorted(set(re.findall(r"arch = (sm_\w+)", sass)))
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            per[cur] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and cur:
            op = m.group(1)
            per[cur]["total"] += 1
            for o in SASS_OPS:
                if op == o or op.startswith(o + "."):
                    per[cur][o] += 1
    names = subprocess.run(["c++filt"], input="\n".join(per), capture_output=True, text=True).stdout.split("\n")
    out = [f"# SASS opcode counts per kernel of libsap_dpsr.so, kernel sources {kernel_tree_hash()}", "",
           "Command: `cuobjdump -sass paper_2106_03452_b200/libsap_dpsr.so` (built by `python -m paper_2106_03452_b200.build`,",
           f"`-gencode arch=compute_100a,code=sm_100a`); architectures in the file: {', '.join(arch)}.  UTMALDG = cp.async.bulk.tensor (TMA),",
           "UBLKCP = cp.async.bulk, SYNCS = mbarrier, FFMA2/FADD2/FMUL2 = packed FP32x2 (sm_100), ACQBULK = griddepcontrol (PDL).  No cuFFT / cuBLAS",
           "symbol is linked (`ldd` shows libcudart only; tests/test_abi_host.py checks it).", "",
           "| kernel | instr | " + " | ".join(SASS_OPS) + " |", "|---|---|" + "---|" * len(SASS_OPS)]
    for (k, c), n in zip(per.items(), names):
        out.append(f"| `{short_name(n)[:70]}` | {c['total']} | " + " | ".join(str(c[o]) for o in SASS_OPS) + " |")
    return "\n".join(out) + "\n"


def main():
    ap = argparse.ArgumentParser()
    sub = ap.add_subparsers(dest="what", required=True)
    a = sub.add_parser("launches"); a.add_argument("csv"); a.add_argument("out"); a.add_argument("--cfg", required=True); a.add_argument("--cmd", required=True)
    b = sub.add_parser("full"); b.add_argument("rep"); b.add_argument("out"); b.add_argument("--cfg", required=True); b.add_argument("--cmd", required=True)
    b.add_argument("--traffic-json"); b.add_argument("--workload")
    c = sub.add_parser("sass"); c.add_argument("out")
    args = ap.parse_args()
    if args.what == "launches":
        Path(args.out).write_text(summarise_launches(args.csv, args.cfg, args.cmd))
    elif args.what == "full":
        md, traffic = summarise_full(args.rep, args.cfg, args.cmd)
        Path(args.out).write_text(md)
        if args.traffic_json:
            p = Path(args.traffic_json)
            doc = json.loads(p.read_text()) if p.exists() else {}
            if doc.get("kernel_sources") != kernel_tree_hash():
                doc = {"kernel_sources": kernel_tree_hash(), "what": "dram__bytes_read.sum + dram__bytes_write.sum per launch (ncu --set full), "
                       "one forward+backward per workload", "workloads": {}}
            doc["workloads"][args.workload or args.cfg] = {"from": args.out, "bytes": traffic_by_label(traffic)}
            p.write_text(json.dumps(doc, indent=1) + "\n")
    else:
        Path(args.out).write_text(summarise_sass())


if __name__ == "__main__":
    main()
