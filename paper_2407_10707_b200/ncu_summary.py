"""Turn an `ncu --set full` report of bench.py into the text summaries kept under profiles/ (no GPU needed: reads the report
with `ncu -i REP --page raw --csv`).

    python -m paper_2407_10707_b200.ncu_summary REP.ncu-rep --md profiles/NAME.md --command "<the full ncu command>" \
        [--counters profiles/ncu_counters.json] [--title "..."]

--md        markdown table: one row per kernel of the report (mean over its launches): time, executed warp instructions, issue
            slot and pipe utilisation, occupancy, DRAM bytes, L2 hit rate
--counters  JSON read by bench.py's `roofline` list: per kernel (bench.py's kernel names) DRAM bytes per launch and executed
            warp instructions per launch, stamped with the hash of csrc/ they were measured on
"""
import argparse
import csv
import json
import os
import subprocess
import sys

from . import build as _build

# CUDA function name (prefix) -> the kernel name rga_profile_read / bench.py uses
NAMES = [("vis_raster_kernel", "vis_raster"), ("vis_shade_kernel", "vis_shade"), ("vis_depth_test_kernel", "vis_depth_test"),
         ("vis_median_kernel", "vis_median"), ("vis_mean_kernel", "vis_mean"), ("shade_paper_kernel", "shade"), ("shade_kernel", "shade"),
         ("skin_kernel", "skin"), ("front_compact_kernel", "front_compact"), ("texel_csr_kernel", "texel_csr"),
         ("env_table_kernel", "env_table"), ("project_kernel", "project"),
         ("tile_scatter_kernel", "tile_scatter"), ("tile_sort_kernel", "tile_sort"),
         ("composite_segment_kernel", "composite_segments"), ("composite_resolve_kernel", "composite_resolve"),
         ("composite_replay_kernel", "composite_replay")]
METRICS = [("gpu__time_duration.sum", "time us", 1e-3), ("smsp__inst_executed.sum", "warp inst", 1.0),
           ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue %", 1.0),
           ("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "fma pipe %", 1.0),
           ("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "alu pipe %", 1.0),
           ("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "xu pipe %", 1.0),
           ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps %", 1.0),
           ("launch__registers_per_thread", "regs", 1.0),
           ("smsp__thread_inst_executed_per_inst_executed.ratio", "lanes/inst", 1.0),
           ("dram__bytes_read.sum", "dram rd MB", None), ("dram__bytes_write.sum", "dram wr MB", None),
           ("lts__t_sector_hit_rate.pct", "L2 hit %", 1.0),
           ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smem conflicts", 1.0)]


def _to_bytes(v, unit):
    u = unit.lower()
    f = {"byte": 1.0, "kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9}.get(u, 1.0)
    return float(v) * f


def _to_us(v, unit):
    u = unit.lower()
    f = {"ns": 1e-3, "nsecond": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "s": 1e6, "second": 1e6}.get(u, 1.0)
    return float(v) * f


def read_report(rep):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(out.splitlines()))
    hdr, units = rows[0], rows[1]
    kn = hdr.index("Kernel Name")
    per = {}
    for r in rows[2:]:
        name = r[kn]
        key = next((k for pre, k in NAMES if pre in name), None)
        if key is None:
            continue
        d = per.setdefault(key, {"launches": 0, "sum": {}, "grid": r[hdr.index("Grid Size")] if "Grid Size" in hdr else "", "block": r[hdr.index("Block Size")] if "Block Size" in hdr else ""})
        d["launches"] += 1
        for m, _, _ in METRICS:
            if m not in hdr:
                continue
            i = hdr.index(m)
            try:
                v = float(r[i].replace(",", ""))
            except ValueError:
                continue
            if m.startswith("dram__bytes"):
                v = _to_bytes(v, units[i])
            elif m == "gpu__time_duration.sum":
                v = _to_us(v, units[i])
            d["sum"][m] = d["sum"].get(m, 0.0) + v
    return per


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--md")
    ap.add_argument("--counters")
    ap.add_argument("--command", default="")
    ap.add_argument("--title", default="")
    ap.add_argument("--frames", type=float, default=1.0, help="frames covered by the capture (launch counts are divided by it)")
    a = ap.parse_args()
    per = read_report(a.report)
    order = sorted(per, key=lambda k: -per[k]["sum"].get("gpu__time_duration.sum", 0.0))
    if a.md:
        with open(a.md, "w") as f:
            f.write("# %s\n\n" % (a.title or os.path.basename(a.report)))
            f.write("Command (committed files only):\n\n    %s\n\n" % a.command)
            f.write("Build: csrc hash `%s`.  Per-kernel MEANS over the launches of the capture (%g frame(s)); a kernel launched twice per frame\n"
                    "(skin: mesh + Gaussians) shows the mean of both.  Times under ncu are serialised and cold-cache: the kernel's SHARE of the\n"
                    "frame is what compares with bench.py's CUDA-event times, not the absolute.\n\n" % (_build.csrc_hash(), a.frames))
            f.write("| kernel | launches/frame | grid x block | " + " | ".join(n for _, n, _ in METRICS) + " |\n")
            f.write("|---|---|---|" + "---|" * len(METRICS) + "\n")
            tot = sum(per[k]["sum"].get("gpu__time_duration.sum", 0.0) for k in order)
            for k in order:
                d = per[k]; n = d["launches"]
                cells = []
                for m, _, _ in METRICS:
                    v = d["sum"].get(m)
                    if v is None:
                        cells.append("-"); continue
                    v /= n
                    if m.startswith("dram__bytes"):
                        cells.append("%.3f" % (v / 1e6))
                    elif m == "smsp__inst_executed.sum" or "conflicts" in m:
                        cells.append("%.3g" % v)
                    else:
                        cells.append("%.1f" % v)
                f.write("| %s | %g | %s x %s | %s |\n" % (k, n / a.frames, d["grid"], d["block"], " | ".join(cells)))
            f.write("\nSum of the kernel times of one frame under ncu: %.1f us.  Shares: %s.\n" % (
                tot / a.frames, ", ".join("%s %.0f %%" % (k, 100 * per[k]["sum"].get("gpu__time_duration.sum", 0.0) / tot) for k in order[:6])))
    if a.counters:
        kern = {}
        for k in order:
            d = per[k]; n = d["launches"]
            lpf = n / a.frames                                   # launches per frame: bench.py's per-kernel time is per frame
            kern[k] = {"dram_bytes": (d["sum"].get("dram__bytes_read.sum", 0.0) + d["sum"].get("dram__bytes_write.sum", 0.0)) / n * lpf,
                       "warp_inst": d["sum"].get("smsp__inst_executed.sum", 0.0) / n * lpf,
                       "ncu_time_us": d["sum"].get("gpu__time_duration.sum", 0.0) / n * lpf}
        json.dump({"source": a.md or a.report, "command": a.command, "csrc_hash": _build.csrc_hash(), "kernels": kern},
                  open(a.counters, "w"), indent=1)
    print("kernels:", ", ".join(order))


if __name__ == "__main__":
    sys.exit(main())
