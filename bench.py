#!/usr/bin/env python
"""bench.py -- relit posed frames/sec of the arXiv 2407.10707 forward render on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (pose_skin -> visibility_raster -> shade_gaussians -> splat_render, all
SURVEY.md 8(a) rows H1..H10) for one frame of one BASELINE.json config, through `rga_render_frame`; seeded synthetic
inputs (synth/).  The contract path is measured: every triangle rasterised (two-sided, no culling),
Gaussians as the generator stores them.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4] [--vis-mode 0|1]
                  [--all-configs 0|1] [--next 0|1] [--no-cpu-baseline]

Prints ONE JSON line (rank 0):
  value / ms_per_step   frames/s of --config (default configs[1], the headline) with inputs resident in HBM, L2 flushed
  e2e                   the same through the C-ABI call with pinned HOST pose / env buffers copied in and the image copied out
  roofline              the dominant kernel of the step: bound, units, work per unit as SURVEY 8(d) states it, CUDA-event time,
                        achieved, MEASURED peak, frac, DRAM bytes per launch from the ncu capture
  roofline_kernels      the same object for every kernel of the frame, largest time first
  configs               all five configs: ms per frame (L2 flushed) + per-kernel and per-stage ms; configs[3] = the 64-pose
                        sequence replayed from one CUDA graph, env map switched per pose, fps = 64 / time
  value_unsorted        the headline frame with the Gaussians in generator (random) order
  frames_in_flight_fps  throughput with 1 / 2 / 3 frames in flight (one avatar handle and stream each; warm L2) -- not `value`
  value_cull_backfaces  the headline frame with the rasteriser's closed-mesh option (A36) -- NOT the contract path
  cpu_baseline          the oracle on this box's host cores: all cores and single thread, per stage
N > 1: replicas only: every rank renders its own frames, no data-path collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "relit posed frames/sec (100k Gaussians, 512x512)"
WORKLOADS = {
    0: "configs[0] tiny: icosphere 642 v / 1,280 f / 2 bones, 2k Gaussians, 8x16 env, 16 dirs @64^2, 64x64",
    1: "configs[1] SMPL-sized: 6,890 v / 13,776 f / 24 bones, 100k Gaussians, 16x32 env, 512 dirs @128^2, 512x512",
    2: "configs[2] high-res: 27,554 v / 55,104 f / 24 bones, 300k Gaussians, 32x64 env, 512 dirs @256^2, 1024x1024",
    3: "configs[3] animation: configs[1] avatar over a 64-pose sequence, 4 env maps switched per pose, 512x512",
    4: "configs[4] stress: 27,554 v / 55,104 f, 1M Gaussians, 32x64 env, 1,024 dirs @256^2, 1920x1080",
}
SM_COUNT, LANES, CLOCK = 148, 128, 1.965e9
FP32_PEAK_DERIVED = 2 * LANES * SM_COUNT * CLOCK / 1e12      # 74.4 TFLOP/s: guide's unit counts x clock (context only)

# Algorithmic work per unit, SURVEY.md 8(d) (issue slots of the FP32/INT lanes; one slot = one FMA-equivalent = 2 flop-eq):
#   H3 ~100 slots per (triangle, direction); H4a ~20 slots per (Gaussian, direction); H5 ~70 flop (45 slots) per evaluated
#   (Gaussian, texel) pair; H10 ~25 slots per evaluated (pixel, list entry).  HBM-bound steps: bytes per unit.
# kernel -> (stage, bound, unit name, work per unit [flop-eq or bytes])
KERNELS = {
    "skin":               ("pose_skin", "hbm", "vertex + Gaussian record", None),
    "vis_raster":         ("visibility", "alu", "(triangle, direction)", 200.0),
    "vis_depth_test":     ("visibility", "alu", "(Gaussian, direction) test", 40.0),
    "vis_median1":        ("visibility", "alu", "(vertex, direction)", None),
    "vis_median2":        ("visibility", "alu", "(vertex, direction)", None),
    "vis_mean":           ("visibility", "alu", "(vertex, direction)", None),
    "env_table":          ("shade", "alu", "texel", None),
    "shade":              ("shade", "alu", "(camera-facing Gaussian, upper-hemisphere texel)", 70.0),
    "vis_shade":          ("shade", "alu", "(Gaussian, direction) test + (Gaussian, texel) BRDF", None),
    "project":            ("splat", "hbm", "Gaussian", 56.0 + 64.0),
    "tile_scatter":       ("splat", "hbm", "duplicate", 8.0 + 8.0),
    "tile_sort":          ("splat", "smem", "list entry", None),
    "composite_T":        ("splat", "alu", "(pixel, list entry)", 50.0),
    "composite_segments": ("splat", "alu", "(pixel, list entry)", 50.0),
    "composite_resolve":  ("splat", "hbm", "pixel", None),
    "composite_replay":   ("splat", "alu", "(pixel, list entry)", None),
}


class ClockSampler:
    """nvidia-smi clocks/throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.stop, self.th = index, [], False, None

    def _run(self):
        while not self.stop:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([t.strip() for t in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def __enter__(self):
        self.th = threading.Thread(target=self._run, daemon=True); self.th.start(); return self

    def __exit__(self, *a):
        self.stop = True; self.th.join(timeout=6)

    def summary(self):
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx[0] if mx else None, "reasons": sorted(reasons),
                "samples": len(self.rows)}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "MEASURED_PEAKS.json"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "B200_PROFILING.md fallback"


def csrc_hash():
    from paper_2407_10707_b200 import build
    return build.csrc_hash()


def ncu_counters():
    """profiles/ncu_counters.json: per-kernel DRAM bytes and executed warp instructions of ONE `ncu --set full` capture of this
    command (written from the capture's raw page), with the csrc hash of the build it was taken on."""
    p = os.path.join(ROOT, "profiles", "ncu_counters.json")
    if not os.path.exists(p):
        return {}, None, False
    d = json.load(open(p))
    return d.get("kernels", {}), d.get("source"), d.get("csrc_hash") == csrc_hash()


def oracle_times(inp, vis_mode, budget_s=12.0):
    """cpu_baseline leg: the oracle as it stands on the host cores -- all cores (OpenMP outer loops) and one thread."""
    from oracle import oracle as orc
    cores = os.cpu_count()
    oav = orc.avatar_load(inp)
    orc.set_num_threads(cores)
    orc.render_frame(oav, inp, vis_mode=vis_mode)
    n, stages, t0 = 0, {}, time.perf_counter()
    while n < 3 or (time.perf_counter() - t0 < budget_s and n < 50):
        orc.render_frame(oav, inp, vis_mode=vis_mode, timings=stages); n += 1
    dt = (time.perf_counter() - t0) / n
    orc.set_num_threads(1)
    st1, t1 = {}, time.perf_counter()
    orc.render_frame(oav, inp, vis_mode=vis_mode, timings=st1)
    dt1 = time.perf_counter() - t1
    orc.set_num_threads(cores)
    return {"value": 1.0 / dt, "unit": "frames/s", "cores": cores, "kind": "oracle",
            "sample": "%d full frames (every step of the path) on all cores, 1 frame on one thread" % n,
            "stage_s": {k: v / n for k, v in stages.items()},
            "single_thread": {"value": 1.0 / dt1, "unit": "frames/s", "cores": 1, "stage_s": st1}}


def run_reference(args, rank):
    """--impl reference: the oracle, as it stands, on the host cores (this tier's reference arm)."""
    if rank != 0:
        return
    from oracle import oracle as orc
    from synth import workloads
    inp = workloads.make(args.config, morton=False)
    cores = os.cpu_count()
    av = orc.avatar_load(inp)
    frames = list(range(len(inp["bone_mats"])))
    for i in range(max(args.warmup, 1)):
        orc.render_frame(av, inp, frame=frames[i % len(frames)], vis_mode=args.vis_mode)
    t0 = time.perf_counter()
    for i in range(args.steps):
        orc.render_frame(av, inp, frame=frames[i % len(frames)], vis_mode=args.vis_mode)
    dt = (time.perf_counter() - t0) / args.steps
    fps = 1.0 / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "vis_mode": args.vis_mode, "vis_cull_backfaces": False},
        "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle",
                         "sample": "%d full frames of %s (every step of the path, OpenMP on outer loops)" % (args.steps, WORKLOADS[args.config][:10])},
        "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


class Bench:
    """One loaded avatar of one config + the timing protocol (CUDA events on the launching stream, L2 flushed between steps)."""

    def __init__(self, cfg, vis_mode, dev, world=1, rank=0, morton=False, flush=None):
        import torch
        from paper_2407_10707_b200 import binding as rga
        from synth import workloads
        self.torch, self.rga, self.cfg, self.vis_mode, self.dev, self.world = torch, rga, cfg, vis_mode, dev, world
        seed = cfg + 1000 * rank if world > 1 else None
        self.inp = inp = workloads.make(cfg, seed=seed, morton=morton)
        cam = inp["camera"]; self.W, self.H = cam["width"], cam["height"]
        self.K, self.R = len(inp["vis_dirs"]), inp["vis_res"]
        t0 = time.perf_counter()
        self.av = rga.Avatar(inp, max_width=self.W, max_height=self.H, max_vis_dirs=self.K, max_vis_res=self.R,
                             max_env_texels=inp["env_rows"] * inp["env_cols"])
        torch.cuda.synchronize(); self.load_ms = (time.perf_counter() - t0) * 1e3
        self.bones = torch.as_tensor(inp["bone_mats"]).to(dev)              # [frames, B, 12]
        self.dirs = torch.as_tensor(inp["vis_dirs"]).to(dev)
        self.envs = torch.as_tensor(inp["env"]).to(dev)                     # [n_env, R, C, 3]
        self.t2d = torch.as_tensor(inp["texel_to_dir"]).to(dev)
        self.img = torch.empty((self.H, self.W, 3), dtype=torch.float32, device=dev)
        self.camc = rga.make_camera(cam)
        self.bias = (inp["depth_bias_texels"], inp["depth_bias_world"], inp["slope_max"])
        self.flush = flush if flush is not None else torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def frame(self, t=0, bones=None, env=None, img=None, cull=False):
        inp = self.inp
        self.av.render(self.bones[t] if bones is None else bones, self.dirs, self.R,
                       self.envs[int(inp["env_of_frame"][t])] if env is None else env, self.t2d, inp["cam_pos"], self.camc, inp["bg"],
                       self.img if img is None else img, vis_mode=self.vis_mode, gamma=inp["gamma"], bias=self.bias, cull_backfaces=cull)

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.torch.distributed.barrier()
        self.torch.cuda.synchronize()

    def timed(self, fn, steps, do_flush=True):
        torch = self.torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        self.barrier()
        for a, b in evs:
            if do_flush:
                self.flush.fill_(1)
            a.record(); fn(); b.record()
        self.barrier()
        return sum(a.elapsed_time(b) for a, b in evs) / steps

    def kernel_times(self, steps, t=0):
        """per-kernel CUDA-event means (the library records an event after each of its kernels; one stream, no overlap)."""
        import numpy as np
        rga = self.rga
        rga.rga_profile_enable(self.av.h, True)
        acc = {}
        for _ in range(steps):
            self.flush.fill_(1)
            self.frame(t)
            for name, ms in rga.rga_profile_read(self.av.h):
                acc.setdefault(name, []).append(ms)
        rga.rga_profile_enable(self.av.h, False)
        return {k: float(np.mean(v)) for k, v in acc.items()}

    def units(self):
        """algorithmic units of each kernel for the frame that was just rendered (counted from its intermediates)."""
        import numpy as np
        inp, av = self.inp, self.av
        gp = av.read("GAUSS_POSED").reshape(-1, 4)[:, :3]; gn = av.read("GAUSS_NORMAL_POSED").reshape(-1, 4)[:, :3]
        front = int((((inp["cam_pos"][None, :] - gp) * gn).sum(1) >= 0).sum())
        rg = av.read("TILE_RANGES").reshape(-1, 2).astype(np.int64)
        D = int(av.read("NUM_DUPLICATES")[0])
        ne = inp["env_rows"] * inp["env_cols"]
        nv, ng, nb = len(inp["vert_pos"]), len(gp), inp["bone_mats"].shape[1]
        nc = av.read("N_CONTRIB").astype(np.int64)
        return {
            "skin": {"units": nv + ng, "bytes": nv * (132 + 24 + 4 * max(nb - 24, 0)) + ng * (176 + 72 + 4 * max(nb - 24, 0))},
            "vis_raster": {"units": len(inp["faces"]) * self.K},
            # inside rga_render_frame the mode-0 depth test runs for the camera-facing Gaussians only
            "vis_depth_test": {"units": front * self.K},
            "shade": {"units": front * ne * 0.5},
            # fused kernel: the depth tests Eq.2 can read (camera-facing Gaussian, direction in its upper hemisphere: 40 flop-eq
            # each) + the BRDF terms (camera-facing Gaussian, upper-hemisphere texel: 70 flop each)
            "vis_shade": {"units": front * self.K * 0.5 + front * ne * 0.5, "flop_eq": front * self.K * 0.5 * 40.0 + front * ne * 0.5 * 70.0},
            "project": {"units": ng},
            "tile_scatter": {"units": D},
            "composite_T": {"units": float(nc.sum())},
            "composite_segments": {"units": float(nc.sum())},
            "_front": front, "_D": D, "_active_tiles": int(((rg[:, 1] - rg[:, 0]) > 0).sum()),
            "_list_max": int((rg[:, 1] - rg[:, 0]).max()), "_pairs_all": float(((rg[:, 1] - rg[:, 0]) * 256).sum()),
            "_pairs_until_stop": float(nc.sum()),
        }

    def close(self):
        self.av.close()


def stage_ms(kern_ms):
    st = {}
    for k, v in kern_ms.items():
        s = KERNELS.get(k, ("other",))[0]
        st[s] = st.get(s, 0.0) + v
    return st


def roofline_list(kern_ms, units, fma_meas, hbm_gbs, hbm_src, with_ncu=True):
    ncu, ncu_src, ncu_ok = ncu_counters() if with_ncu else ({}, None, False)
    out = []
    for k, ms in sorted(kern_ms.items(), key=lambda kv: -kv[1]):
        stage, bound, unit_name, work = KERNELS.get(k, ("other", "alu", "", None))
        u = units.get(k)
        o = {"kernel": k, "stage": stage, "bound": bound, "kernel_ms": ms}
        if u is not None and bound == "hbm" and ("bytes" in u or work):
            byts = u.get("bytes", u["units"] * (work or 0))
            o.update(units_per_launch=u["units"], unit_of_work=unit_name, bytes_per_launch=byts, achieved=byts / (ms * 1e-3) / 1e9,
                     peak=hbm_gbs, peak_source=hbm_src, unit="GB/s")
            o["frac"] = o["achieved"] / o["peak"]
        elif u is not None and (work or "flop_eq" in u) and bound == "alu":
            flop_eq = u.get("flop_eq", u["units"] * (work or 0.0))
            ach = flop_eq / (ms * 1e-3) / 1e12
            o.update(units_per_launch=u["units"], unit_of_work=unit_name, flop_eq_per_unit=flop_eq / u["units"], flop_eq_per_launch=flop_eq,
                     achieved=ach, peak=fma_meas,
                     peak_source="register-resident FFMA chains measured in this run (rga_measure_fp32_peak)",
                     peak_derived=FP32_PEAK_DERIVED, unit="TFLOP/s", frac=ach / fma_meas if fma_meas > 0 else None)
        else:
            o.update(achieved=None, peak=None, frac=None, unit=None, note="latency / launch bound helper kernel: no work model")
        c = ncu.get(k)
        if c and ncu_ok:
            o["traffic"] = c.get("dram_bytes"); o["traffic_source"] = ncu_src
            if c.get("warp_inst"):
                o["issue_slots"] = {"executed_warp_inst": c["warp_inst"],
                                    "frac_of_issue_peak": c["warp_inst"] / (ms * 1e-3) / (SM_COUNT * 4 * CLOCK)}
        else:
            o["traffic"] = None
            if c and not ncu_ok:
                o["traffic_note"] = "profiles/ncu_counters.json was captured on another build of csrc/ (hash mismatch): not quoted"
        out.append(o)
    return out


def bench_config(cfg, vis_mode, dev, steps, warmup, flush, fma_meas):
    """One entry of `configs`: ms per frame (L2 flushed), per-kernel / per-stage ms; configs[3]: the 64-pose graph replay."""
    import torch
    b = Bench(cfg, vis_mode, dev, morton=False, flush=flush)
    rga = b.rga
    nfr = len(b.inp["bone_mats"])
    for i in range(warmup):
        b.frame(i % nfr)
    rga.rga_check(b.av.h)
    out = {"workload": WORKLOADS[cfg], "avatar_load_ms": b.load_ms}
    if nfr > 1:
        # SURVEY 8(d) timing protocol: the whole pose sequence captured once as a CUDA graph (re-skinning, re-visibility,
        # env map switched per pose), replayed; steady-state fps = frames / time
        g = torch.cuda.CUDAGraph(); st = torch.cuda.Stream(device=dev)
        st.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(st):
            with torch.cuda.graph(g, stream=st):
                for t in range(nfr):
                    b.frame(t)
        torch.cuda.current_stream().wait_stream(st)
        g.replay(); torch.cuda.synchronize()
        reps = max(2, min(steps, 10))
        ms_seq = b.timed(g.replay, reps)
        rga.rga_check(b.av.h)
        out.update(protocol="%d-pose sequence in ONE CUDA graph, env map switched per pose, L2 flushed between replays" % nfr,
                   ms_per_sequence=ms_seq, ms_per_frame=ms_seq / nfr, fps=nfr * 1e3 / ms_seq, envs_used=len(set(int(e) for e in b.inp["env_of_frame"])))
        ms_single = b.timed(lambda: b.frame(7), max(3, min(steps, 20)))
        out["ms_per_frame_single_call_flushed"] = ms_single
    else:
        ms = b.timed(b.frame, steps)
        out.update(protocol="rga_render_frame per step, L2 flushed between steps", ms_per_frame=ms, fps=1e3 / ms)
    km = b.kernel_times(max(3, min(steps, 10)))
    u = b.units()
    pk, pk_src = peaks()
    rl = roofline_list(km, u, fma_meas, pk["hbm_gbs"], pk_src, with_ncu=False)
    out["roofline"] = [{k: r.get(k) for k in ("kernel", "bound", "kernel_ms", "units_per_launch", "flop_eq_per_unit", "bytes_per_launch", "achieved",
                                            "peak", "unit", "frac")} for r in rl if r.get("frac") is not None]
    out.update(kernel_ms=km, stage_ms=stage_ms(km), duplicates=u["_D"], camera_facing_gaussians=u["_front"], active_tiles=u["_active_tiles"],
               longest_tile_list=u["_list_max"], blend_pairs_until_stop=u["_pairs_until_stop"], blend_pairs_all=u["_pairs_all"])
    rga.rga_check(b.av.h)
    b.close()
    del b
    torch.cuda.empty_cache()
    return out


def next_rows(b, steps):
    """SURVEY 8(f) rows, reported beside the metric (not part of it); same timing protocol."""
    import numpy as np
    import torch
    from synth import workloads
    rga, av, inp, dev, camc, img = b.rga, b.av, b.inp, b.dev, b.camc, b.img
    bones, env, t2d, dirs = b.bones[0], b.envs[0], b.t2d, b.dirs
    out = {}
    NV = 4

    def pose_with_views():
        rga.pose_skin(av.h, bones)
        rga.visibility_raster(av.h, dirs, b.R, b.vis_mode, b.bias[0], b.bias[1], b.bias[2])
        for _ in range(NV):
            rga.shade_gaussians(av.h, env, inp["cam_pos"], t2d, inp["gamma"], True)
            rga.splat_render(av.h, camc, inp["bg"], img)
    for _ in range(3):
        pose_with_views()
    ms_views = b.timed(pose_with_views, max(steps // 4, 5))
    out["amortised"] = {"views_per_pose": NV, "views_per_s": NV * 1e3 / ms_views, "ms_per_pose": ms_views}
    b.frame()
    dLdI = torch.as_tensor(workloads.make_image_cotangent(1, camc.width, camc.height)).to(dev)
    ng_all, nv_all, nb_all = len(inp["gauss_pos"]), len(inp["vert_pos"]), inp["bone_mats"].shape[1]
    d_col = torch.empty((ng_all, 3), device=dev); d_op = torch.empty((ng_all,), device=dev)
    d_x = torch.empty((ng_all, 3), device=dev); d_cov = torch.empty((ng_all, 6), device=dev)
    run_bwd = lambda: rga.splat_backward(av.h, camc, inp["bg"], img, dLdI, d_col, d_op, d_x, d_cov)
    for _ in range(3):
        run_bwd()
    out["splat_backward"] = {"ms": b.timed(run_bwd, 20)}
    ne_all = int(env.shape[0] * env.shape[1])
    sb = dict(out_dalbedo=torch.empty((ng_all, 3), device=dev), out_drough=torch.empty((ng_all,), device=dev),
              out_dspec=torch.empty((ng_all,), device=dev), out_dnormal=torch.empty((ng_all, 3), device=dev),
              out_dpos=torch.empty((ng_all, 3), device=dev), out_denv=torch.empty((ne_all, 3), device=dev))
    run_sb = lambda: rga.shade_backward(av.h, env, inp["cam_pos"], d_col, texel_to_dir=t2d, gamma=inp["gamma"], use_visibility=True, **sb)
    for _ in range(3):
        run_sb()
    out["shade_backward"] = {"ms": b.timed(run_sb, 20), "gaussians_with_gradient": int((d_col.abs().sum(1) > 0).sum().item())}
    _, tgt_np = workloads.make_image_pair(1, camc.width, camc.height)
    tgt_d = torch.as_tensor(tgt_np).to(dev); loss_d = torch.zeros(3, device=dev)
    run_il = lambda: rga.image_loss(av.h, img, tgt_d, 0.2, loss_d, dLdI)
    for _ in range(3):
        run_il()
    out["image_loss"] = {"ms": b.timed(run_il, 20)}
    rg = dict(out_losses=torch.zeros(4, device=dev), out_dalbedo=torch.empty((nv_all, 3), device=dev), out_drough=torch.empty(nv_all, device=dev),
              out_dspec=torch.empty(nv_all, device=dev), out_dgauss_pos=torch.empty((ng_all, 3), device=dev),
              out_ddisp=torch.empty((nv_all, 3), device=dev), out_dscale=torch.empty((ng_all, 3), device=dev))
    run_rg = lambda: rga.regularisers(av.h, 0.005, **rg)
    for _ in range(3):
        run_rg()
    out["regularisers"] = {"ms": b.timed(run_rg, 20)}
    pb_out = {"d_gauss_pos": torch.empty((ng_all, 3), device=dev), "d_gauss_quat": torch.empty((ng_all, 4), device=dev),
              "d_gauss_scale": torch.empty((ng_all, 3), device=dev), "d_bones": torch.empty((nb_all, 12), device=dev),
              "d_vert_disp": torch.empty((nv_all, 3), device=dev), "d_vert_normal": torch.empty((nv_all, 3), device=dev),
              "d_vert_albedo": torch.empty((nv_all, 3), device=dev), "d_vert_rough": torch.empty(nv_all, device=dev),
              "d_vert_spec": torch.empty(nv_all, device=dev)}
    pb_in = {"d_mean": d_x, "d_mean2": sb["out_dpos"], "d_normal": sb["out_dnormal"], "d_cov": d_cov, "d_albedo": sb["out_dalbedo"],
             "d_rough": sb["out_drough"], "d_spec": sb["out_dspec"]}
    run_pb = lambda: rga.pose_backward(av.h, bones, pb_in, pb_out)
    for _ in range(3):
        run_pb()
    ms_pb = b.timed(run_pb, 20)

    def run_chain():
        run_il(); run_bwd(); run_sb(); run_pb()
    for _ in range(3):
        run_chain()
    out["train_backward"] = {"pose_backward_ms": ms_pb, "backward_chain_ms": b.timed(run_chain, 20),
                             "note": "image_loss + splat_backward + shade_backward + pose_backward of the rendered view"}
    mlp = workloads.make_disp_mlp(seed=1)
    mlp_d = {k: (torch.as_tensor(v).to(dev) if isinstance(v, np.ndarray) else v) for k, v in mlp.items()}
    run_mlp = lambda: rga.displacement_mlp(av.h, mlp_d, mlp_d["theta"])
    for _ in range(3):
        run_mlp()
    rga.rga_profile_enable(av.h, True)
    mlp_t = []
    for _ in range(20):
        run_mlp()
        mlp_t += [t for name, t in rga.rga_profile_read(av.h) if name == "disp_mlp"]
    rga.rga_profile_enable(av.h, False)
    mlp_flop = 2.0 * nv_all * (2 * mlp["n_freq"] * 256 + 3 * 256 * 256 + 3 * 256)
    mlp_ms = float(np.mean(mlp_t))
    pk, _ = peaks()
    tf32_peak = pk.get("bf16_tflops", 1590.0) * (1.1 / 2.25)          # measured bf16 peak x the guide's nominal tf32 : bf16 ratio
    out["disp_mlp"] = {"kernel": "disp_mlp", "bound": "tensor", "ms": mlp_ms, "achieved": mlp_flop / (mlp_ms * 1e-3) / 1e12, "peak": tf32_peak,
                       "unit": "TFLOP/s", "frac": mlp_flop / (mlp_ms * 1e-3) / 1e12 / tf32_peak, "dtype": "tf32 operands, f32 accumulate"}
    gp = torch.as_tensor(inp["gauss_pos"]).to(dev)
    for _ in range(3):
        rga.gaussians_update(av.h, gp)
    out["gaussians_update_ms"] = b.timed(lambda: rga.gaussians_update(av.h, gp), 20)
    n_dens = 65536
    d_rnd = torch.randint(-2 ** 31, 2 ** 31 - 1, (3 * n_dens,), dtype=torch.int32, device=dev, generator=torch.Generator(dev).manual_seed(5))
    d_pos = torch.empty((n_dens, 3), dtype=torch.float32, device=dev); d_cnt = torch.zeros(1, dtype=torch.int32, device=dev)
    for _ in range(3):
        rga.densify_density(av.h, 12.0, 0.25, d_rnd, d_pos, None, d_cnt)
    out["densify_density"] = {"ms": b.timed(lambda: rga.densify_density(av.h, 12.0, 0.25, d_rnd, d_pos, None, d_cnt), 20),
                              "d0": 12.0, "p0": 0.25, "added": int(d_cnt.item())}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4], help="BASELINE.json config of the main line (default 1, the headline)")
    ap.add_argument("--vis-mode", type=int, default=0, help="0 = depth test (north_star, default), 1 = paper filters")
    ap.add_argument("--all-configs", type=int, default=1, help="1 (default): also time all five configs -> `configs`")
    ap.add_argument("--next", type=int, default=1, help="1 (default): also time the SURVEY 8(f) rows")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        if args.steps == 200 and args.warmup == 20:
            args.steps, args.warmup = 10, 1
        return run_reference(args, rank)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2407_10707_b200 import binding as rga
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    dev = torch.device("cuda", local)
    cfg = args.config
    b = Bench(cfg, args.vis_mode, dev, world=world, rank=rank, morton=False)
    inp, av, W, H = b.inp, b.av, b.W, b.H
    nfr = len(inp["bone_mats"])
    steps = args.steps if cfg in (0, 1, 3) else max(10, min(args.steps, 40))
    it = [0]

    def frame():                                                # config 3 walks its pose sequence; the others have one pose
        b.frame(it[0] % nfr); it[0] += 1

    for _ in range(args.warmup):
        frame()
    rga.rga_check(av.h)
    l0 = rga.rga_launch_count(av.h)
    cs = ClockSampler(local); cs.__enter__()                     # sampled through every timed pass below
    ms = b.timed(frame, steps)
    launches = (rga.rga_launch_count(av.h) - l0) / steps
    ms_warm = b.timed(frame, steps, do_flush=False)

    # end to end: host (pinned) pose + env in, image out, every step, through the same C-ABI call
    h_bones = torch.as_tensor(inp["bone_mats"][0]).pin_memory(); h_env = torch.as_tensor(inp["env"][0]).pin_memory()
    h_img = torch.empty((H, W, 3), dtype=torch.float32).pin_memory()
    d_bones = torch.empty_like(b.bones[0]); d_env = torch.empty_like(b.envs[0])

    def frame_e2e():
        d_bones.copy_(h_bones, non_blocking=True); d_env.copy_(h_env, non_blocking=True)
        b.frame(0, bones=d_bones, env=d_env)
        h_img.copy_(b.img, non_blocking=True)
    for _ in range(3):
        frame_e2e()
    ms_e2e = b.timed(frame_e2e, steps)

    # the documented viewer loop: the image read-back of step i on a copy stream beside step i+1 (two image buffers).
    # Reported as e2e.pipelined_value; e2e.value stays the serial number above.
    copy_stream = torch.cuda.Stream(device=dev)
    imgs = [torch.empty_like(b.img) for _ in range(2)]
    h_imgs = [torch.empty((H, W, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    copied = [None, None]

    def run_pipelined(n):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        last_copy = None
        b.barrier()
        for i, (a, e) in enumerate(evs):
            b.flush.fill_(1)
            a.record()
            if copied[i & 1] is not None:
                torch.cuda.current_stream().wait_event(copied[i & 1])     # buffer i&1 has been read back
            d_bones.copy_(h_bones, non_blocking=True); d_env.copy_(h_env, non_blocking=True)
            b.frame(0, bones=d_bones, env=d_env, img=imgs[i & 1])
            e.record()
            copy_stream.wait_event(e)
            with torch.cuda.stream(copy_stream):
                h_imgs[i & 1].copy_(imgs[i & 1], non_blocking=True)
                copied[i & 1] = torch.cuda.Event(enable_timing=True); copied[i & 1].record()
                last_copy = copied[i & 1]
        b.barrier(); copy_stream.synchronize()
        tail = max(evs[-1][1].elapsed_time(last_copy), 0.0)                # the last read-back is not hidden by a next step
        return (sum(a.elapsed_time(e) for a, e in evs) + tail) / n
    run_pipelined(3)
    ms_e2e_pipe = run_pipelined(steps)

    kern_ms = b.kernel_times(steps)
    rga.rga_check(av.h)
    t_end = time.time() + 1.0                                      # at least a second of load for the sampler
    while time.time() < t_end or len(cs.rows) < 3:
        for _ in range(50):
            frame()
        torch.cuda.synchronize()
        if time.time() > t_end + 5.0:
            break
    cs.__exit__(); clocks = cs.summary()
    b.frame(0)
    units = b.units()
    pk, pk_src = peaks()
    fma_meas = rga.rga_measure_fp32_peak()
    roofline = roofline_list(kern_ms, units, fma_meas, pk["hbm_gbs"], pk_src)

    # the rasteriser's closed-mesh option (reading A36) -- NOT the contract path, reported beside it
    for _ in range(3):
        b.frame(0, cull=True)
    ms_cull = b.timed(lambda: b.frame(0, cull=True), max(steps // 4, 10))
    extra = next_rows(b, steps) if (args.next and world == 1 and cfg == 1) else {}
    b.close()

    ms_sorted = None
    if world == 1:                                                 # the same frame with the Gaussians in spatial (Morton) order
        bs = Bench(cfg, args.vis_mode, dev, morton=True, flush=b.flush)
        for _ in range(args.warmup):
            bs.frame(0)
        ms_sorted = bs.timed(lambda: bs.frame(0), max(steps // 2, 10))
        bs.close()

    # Throughput with more than one frame in flight (offline rendering of independent frames, several avatars on one GPU): two /
    # three avatar handles, each on its own stream, frames issued round robin, no L2 flush (compare with warm_l2_fps).  The
    # frame's latency-bound phases (skinning, the blend's fold and replay) overlap the other frame's big kernels.  NOT `value`:
    # a viewer shows frames one after the other.
    in_flight = None
    if world == 1 and cfg in (0, 1, 3):
        insts = [Bench(cfg, args.vis_mode, dev, flush=b.flush) for _ in range(3)]
        streams = [torch.cuda.Stream(device=dev) for _ in range(3)]

        def run_in_flight(k, n):
            torch.cuda.synchronize()
            a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for st in streams[:k]:
                st.wait_stream(torch.cuda.current_stream())
            for i in range(n):
                with torch.cuda.stream(streams[i % k]):
                    insts[i % k].frame(0)
            for st in streams[:k]:
                torch.cuda.current_stream().wait_stream(st)
            e.record(); torch.cuda.synchronize()
            return n / (a.elapsed_time(e) * 1e-3)
        in_flight = {"note": "avatar handles on their own streams, frames issued round robin, warm L2; whole-run CUDA-event time"}
        for k in (1, 2, 3):
            run_in_flight(k, 30)
            in_flight[str(k)] = run_in_flight(k, max(steps, 100))
        for x in insts:
            x.close()

    from paper_2407_10707_b200 import replica
    ms, ms_e2e, ms_warm = replica.max_over_ranks([ms, ms_e2e, ms_warm], device=dev)      # slowest rank sets the job time
    out = {
        "metric": METRIC, "value": world * 1e3 / ms, "unit": "frames/s", "n_gpus": world, "steps": steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOADS[cfg], "vis_mode": args.vis_mode, "vis_cull_backfaces": False,
                   "gaussian_order": "generator order (random surface points, unsorted)",
                   "l2": "flushed between steps (256 MiB fill)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU", "paper_context": "6.9 fps on RTX 4090 (PAPER.md:314)"},
        "clocks": clocks, "gpu_launches": int(round(launches * steps)), "gpu_launches_per_step": launches,
        "e2e": {"value": world * 1e3 / ms_e2e, "unit": "frames/s", "h2d_bytes_per_step": int(h_bones.numel() * 4 + h_env.numel() * 4),
                "d2h_bytes_per_step": int(h_img.numel() * 4),
                "pipelined_value": world * 1e3 / ms_e2e_pipe,
                "pipelined_note": "the documented viewer loop: image read-back of step i on a copy stream beside step i+1"},
        "roofline": dict(roofline[0], note="the dominant kernel of the step; every kernel of the frame is in roofline_kernels"),
        "roofline_kernels": roofline, "kernel_ms": kern_ms, "stage_ms": stage_ms(kern_ms), "warm_l2_fps": world * 1e3 / ms_warm,
        "avatar_load_ms": b.load_ms,
        "value_unsorted": world * 1e3 / ms, "value_spatially_sorted_input": (1e3 / ms_sorted) if ms_sorted else None,
        "value_cull_backfaces": world * 1e3 / ms_cull, "frames_in_flight_fps": in_flight,
        "workload_stats": {k[1:]: v for k, v in units.items() if k.startswith("_")},
    }
    out.update(extra)
    if rank == 0 and world == 1 and args.all_configs:
        flush = b.flush
        out["configs"] = {}
        for c in range(5):
            out["configs"][str(c)] = bench_config(c, args.vis_mode, dev, max(5, min(args.steps, 20 if c in (2, 4) else 50)), 3, flush, fma_meas)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = oracle_times(inp, args.vis_mode)     # the oracle is imported only here, after every timed region
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
