"""Markdown tables from a bench.py JSON line (the tables of BASELINE.md "Results" are this module's output, so that the
committed numbers can be re-derived from the committed JSON).

    python -m paper_2407_10707_b200.report profiles/r02_bench.json
"""
import json
import sys


def _f(v, nd=3):
    return "-" if v is None else ("%." + str(nd) + "f") % v


def main():
    d = json.load(open(sys.argv[1]))
    print("Headline (%s):" % d["config"]["workload"])
    print()
    print("| quantity | value |")
    print("|---|---|")
    print("| `value` (frames/s, inputs in HBM, L2 flushed) | %.1f (%.4f ms per frame, %d steps) |" % (d["value"], d["ms_per_step"], d["steps"]))
    print("| `e2e.value` (host pose + env in, image out, serial) | %.1f |" % d["e2e"]["value"])
    print("| `e2e.pipelined_value` (read-back on a copy stream) | %.1f |" % d["e2e"]["pipelined_value"])
    print("| `warm_l2_fps` (no L2 flush) | %.1f |" % d["warm_l2_fps"])
    print("| `value_spatially_sorted_input` (same frame, Gaussians pre-sorted) | %s |" % _f(d.get("value_spatially_sorted_input"), 1))
    fl = d.get("frames_in_flight_fps")
    if fl:
        print("| `frames_in_flight_fps` (1 / 2 / 3 avatar handles on their own streams, warm L2; not the metric) | %.1f / %.1f / %.1f |" % (fl["1"], fl["2"], fl["3"]))
    print("| `value_cull_backfaces` (closed-mesh option, NOT the contract path) | %.1f |" % d["value_cull_backfaces"])
    print("| kernels launched per frame | %s |" % _f(d.get("gpu_launches_per_step"), 0))
    print("| `avatar_load` (once) | %.1f ms |" % d["avatar_load_ms"])
    print("| SM clock under load / max, throttle reasons | %s / %s MHz, %s |" % (d["clocks"]["sm_mhz"], d["clocks"]["sm_max_mhz"], d["clocks"]["reasons"]))
    cb = d.get("cpu_baseline")
    if cb:
        print("| oracle, %d host cores | %.2f frames/s (%s) |" % (cb["cores"], cb["value"], ", ".join("%s %.3f s" % kv for kv in cb["stage_s"].items())))
        st = cb["single_thread"]
        print("| oracle, 1 thread | %.3f frames/s (%s) |" % (st["value"], ", ".join("%s %.3f s" % kv for kv in st["stage_s"].items())))
    print()
    print("Per-kernel roofline of the headline frame (`roofline_kernels`; `roofline` is its first row; CUDA-event time per kernel, one stream):")
    print()
    print("| kernel | stage | bound | time us | units | work per unit | achieved | peak (measured) | frac | DRAM MB (ncu) | issue slots busy |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for r in (d.get("roofline_kernels") or d["roofline"]):
        unit = r.get("unit") or ""
        wpu = r.get("flop_eq_per_unit")
        if wpu is None and r.get("bytes_per_launch") and r.get("units_per_launch"):
            wpu = r["bytes_per_launch"] / r["units_per_launch"]
        tr = r.get("traffic")
        isl = (r.get("issue_slots") or {}).get("frac_of_issue_peak")
        print("| %s | %s | %s | %.1f | %s | %s | %s | %s | %s | %s | %s |" % (
            r["kernel"], r["stage"], r["bound"], r["kernel_ms"] * 1e3,
            "-" if r.get("units_per_launch") is None else "%.3g" % r["units_per_launch"],
            "-" if wpu is None else ("%.0f %s" % (wpu, "B" if r["bound"] == "hbm" else "flop-eq")),
            "-" if r.get("achieved") is None else "%.1f %s" % (r["achieved"], unit),
            "-" if r.get("peak") is None else "%.1f" % r["peak"],
            "-" if r.get("frac") is None else "%.3f" % r["frac"],
            "-" if tr is None else "%.2f" % (tr / 1e6), "-" if isl is None else "%.2f" % isl))
    if "configs" in d:
        print()
        print("All five configs (same run, same protocol; config 3 = 64-pose CUDA-graph replay):")
        print()
        print("| config | ms per frame | frames/s | pose_skin | visibility | shade | splat (stage ms, one stream) | duplicates D | longest list | blend pairs until stop / walked |")
        print("|---|---|---|---|---|---|---|---|---|---|")
        for c, v in d["configs"].items():
            st = v["stage_ms"]
            print("| %s | %.3f | %.1f | %.3f | %.3f | %.3f | %.3f | %d | %d | %.3g / %.3g |" % (
                v["workload"].split(":")[0], v["ms_per_frame"], v["fps"], st.get("pose_skin", 0), st.get("visibility", 0), st.get("shade", 0),
                st.get("splat", 0), v["duplicates"], v["longest_tile_list"], v["blend_pairs_until_stop"], v["blend_pairs_all"]))
        print()
        print("Per-kernel us per config:")
        print()
        names = []
        for v in d["configs"].values():
            for k in v["kernel_ms"]:
                if k not in names:
                    names.append(k)
        print("| kernel | " + " | ".join("cfg%s" % c for c in d["configs"]) + " |")
        print("|---|" + "---|" * len(d["configs"]))
        for k in names:
            print("| %s | %s |" % (k, " | ".join("%.1f" % (v["kernel_ms"].get(k, 0.0) * 1e3) for v in d["configs"].values())))
        print()
        print("Per-kernel roofline fraction per config (achieved / measured peak; work per unit as in the headline table):")
        print()
        kn = []
        for v in d["configs"].values():
            for r in v.get("roofline", []):
                if r["kernel"] not in kn:
                    kn.append(r["kernel"])
        print("| kernel | " + " | ".join("cfg%s" % c for c in d["configs"]) + " |")
        print("|---|" + "---|" * len(d["configs"]))
        for k in kn:
            cells = []
            for v in d["configs"].values():
                r = next((r for r in v.get("roofline", []) if r["kernel"] == k), None)
                cells.append("-" if r is None else "%.3f (%.1f %s)" % (r["frac"], r["achieved"], r["unit"]))
            print("| %s | %s |" % (k, " | ".join(cells)))
    nx = [k for k in ("amortised", "disp_mlp", "gaussians_update_ms", "densify_density", "image_loss", "splat_backward", "shade_backward",
                      "regularisers", "train_backward") if k in d]
    if nx:
        print()
        print("SURVEY 8(f) rows (beside the metric): " + "; ".join("%s %s" % (k, json.dumps(d[k])) for k in nx))


if __name__ == "__main__":
    main()
