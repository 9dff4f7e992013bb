"""Shared helper of the GPU parity tests: run the CUDA path through the C-ABI binding and the oracle on the same seeded
inputs and compare every stage.  Integer / index / bit outputs must be identical; radiance, colour and image obey the
north_star tolerances (max-abs 2e-3, mean-abs 2e-4 on [0,1] values)."""
import numpy as np

IMG_MAX, IMG_MEAN = 2e-3, 2e-4


def run_gpu(inp, vis_mode=0, frame=0, keep_maps=True, use_visibility=True, max_duplicates=0, camera=None):
    import torch
    from paper_2407_10707_b200 import binding as rga
    cam = camera or inp["camera"]
    W, H = cam["width"], cam["height"]
    dev = "cuda"
    av = rga.Avatar(inp, max_width=W, max_height=H, max_vis_dirs=len(inp["vis_dirs"]), max_vis_res=inp["vis_res"],
                    max_env_texels=inp["env_rows"] * inp["env_cols"], max_duplicates=max_duplicates)
    bones = torch.as_tensor(inp["bone_mats"][frame]).to(dev)
    dirs = torch.as_tensor(inp["vis_dirs"]).to(dev)
    env = torch.as_tensor(inp["env"][inp["env_of_frame"][frame]]).to(dev)
    t2d = torch.as_tensor(inp["texel_to_dir"]).to(dev)
    img = torch.empty((H, W, 3), dtype=torch.float32, device=dev)
    rga.pose_skin(av.h, bones)
    if use_visibility:
        rga.visibility_raster(av.h, dirs, inp["vis_res"], vis_mode, inp["depth_bias_texels"], inp["depth_bias_world"],
                              inp["slope_max"], keep_maps, cull_backfaces=bool(inp.get("vis_cull_backfaces", False)))
    rga.shade_gaussians(av.h, env, inp["cam_pos"], t2d, inp["gamma"], use_visibility)
    rga.splat_render(av.h, cam, inp["bg"], img)
    rga.rga_check(av.h)
    torch.cuda.synchronize()
    return av, img.cpu().numpy()


def facing_split(inp, o, cam_pos=None):
    """(kept, culled) masks of the Gaussians w.r.t. the camera-facing test of rga_render_frame / shade_gaussians
    (PAPER.md:101), with a guard band around 0 in which neither is asserted."""
    cp = inp["cam_pos"] if cam_pos is None else cam_pos
    wo = cp[None, :].astype(np.float64) - o["gauss_posed"]
    f = (wo * o["gauss_normal_posed"]).sum(1) / np.linalg.norm(wo, axis=1)
    return f > 1e-3, f < -1e-3


def check_frame_visbits(inp, o, vb, cam_pos=None, fused=True):
    """Visibility words written by rga_render_frame's fused depth-test + shading kernel (mode 0).  It tests a (Gaussian,
    direction) pair only when Eq.2 can read the result: the Gaussian faces the camera and the direction d
    has a texel k with w_i^k . n > 0 (v_g[k] max(0, w_i . n)), decided conservatively as
    n . w_d > -eps_d with eps_d = the largest chord |w_k - w_d| over the texels that read d, + 1e-3.  Pairs that must be
    tested have to equal the oracle's bit; pairs that cannot be tested have to be 0; a 1e-5 band around the rule is free."""
    from oracle import oracle as orc
    ng, K = len(inp["gauss_pos"]), len(inp["vis_dirs"])
    kept, culled = facing_split(inp, o, cam_pos)
    wk, _ = orc.env_table(inp["env_rows"], inp["env_cols"])
    t2d = inp["texel_to_dir"]
    dirs = inp["vis_dirs"].astype(np.float64)
    eps = np.full(K, -4.0)
    chord = np.linalg.norm(wk - dirs[t2d], axis=1)
    np.maximum.at(eps, t2d, chord + 1e-3)
    got = ((vb[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(ng, -1)[:, :K].astype(bool)
    ref = ((o["visbits"][:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(ng, -1)[:, :K].astype(bool)
    assert not got[culled].any(), "visibility words of Gaussians facing away from the camera"
    n_checked = 0
    for a in range(0, ng, 100_000):                                      # chunks keep the [ng, K] cosine table small
        b = min(ng, a + 100_000)
        cs = o["gauss_normal_posed"][a:b].astype(np.float64) @ dirs.T
        must = kept[a:b, None] & (cs > -eps[None, :] + 1e-5)
        never = cs < -eps[None, :] - 1e-5
        assert np.array_equal(got[a:b][must], ref[a:b][must]), "visibility bits of tested (Gaussian, direction) pairs"
        if fused:                                                         # the two-kernel fallback (tables beyond shared memory) tests every direction
            assert not got[a:b][never].any(), "visibility bits of directions Eq.2 cannot read"
        n_checked += int(must.sum())
    # (a grid of one or two directions can stand behind every camera-facing Gaussian: sweep seed 54952, one light opposite the viewer)
    assert n_checked > 0 or K < 8
    return n_checked


def compare_all(inp, av, img, orc_av, o, vis_mode, use_visibility=True, report=None, frame_call=False, flag_per_pair=None, fused=True):
    """Assert stage-by-stage parity.  `o` is oracle.render_frame's dict, `orc_av` oracle.avatar_load's.
    frame_call: the frame came from rga_render_frame, whose mode-0 depth test skips Gaussians that face away from the
    camera (their bits are never read): visibility bits are compared on the kept Gaussians and must be 0 on the culled."""
    rep = report if report is not None else {}
    ng, nv = len(inp["gauss_pos"]), len(inp["vert_pos"])
    K, R = len(inp["vis_dirs"]), inp["vis_res"]
    words = (K + 31) // 32
    rd = av.read
    eq = np.array_equal

    # L0
    assert eq(rd("KNN_G").reshape(ng, -1), orc_av["knn_g"]), "knn_g"
    assert eq(rd("KNN_V").reshape(nv, -1), orc_av["knn_v"]), "knn_v"
    assert eq(rd("UBAR_G").reshape(ng, -1), orc_av["ubar_g"]), "ubar_g"
    st = rd("GAUSS_STATIC").reshape(ng, 16)
    assert eq(st[:, 0:3], inp["gauss_pos"] + orc_av["disp_g"]), "xbar_g"
    assert eq(st[:, 4:7], orc_av["normal_g"]), "normal_g"
    assert eq(st[:, 8:11], orc_av["albedo_g"]) and eq(st[:, 11], orc_av["rough_g"]) and eq(st[:, 12], orc_av["spec_g"]), "materials"
    assert eq(rd("GAUSS_SKIN_W").reshape(ng, -1), orc_av["skin_w_g"]), "skin_w_g"
    # H1/H2 (bit-exact fp32)
    assert eq(rd("VERT_POSED").reshape(nv, 4)[:, :3], o["vert_posed"]), "vert_posed"
    assert eq(rd("VERT_NORMAL_POSED").reshape(nv, 4)[:, :3], o["vert_normal_posed"]), "vert_normal_posed"
    assert eq(rd("GAUSS_POSED").reshape(ng, 4)[:, :3], o["gauss_posed"]), "gauss_posed"
    assert eq(rd("GAUSS_NORMAL_POSED").reshape(ng, 4)[:, :3], o["gauss_normal_posed"]), "gauss_normal_posed"
    assert eq(rd("GAUSS_COV").reshape(ng, 6), o["cov6"]), "cov6"
    win = rd("WINDOW")
    assert eq(win[:3], o["win_c"]) and win[3] == o["win_r"], "window"
    # H3/H4
    if use_visibility:
        assert eq(rd("ZMAP").reshape(K, R, R), o["zmap"]), "zmap"
        ids = rd("IDMAP")
        if ids.size:
            assert eq(ids.reshape(K, R, R), o["idmap"]), "idmap"
        if vis_mode == 0:
            vb = rd("VISBITS").reshape(ng, words)
            if frame_call:
                rep["visbits_checked"] = check_frame_visbits(inp, o, vb, fused=fused)
            else:
                assert eq(vb, o["visbits"]), "visbits"
        else:
            assert eq(rd("VCOUNT").reshape(nv, K), o["vcount"]), "vcount"
    # H6 (bit-exact)
    assert eq(rd("TOUCHED"), o["touched"]), "touched"
    assert eq(rd("RECT").reshape(ng, 4), o["rect"]), "rect"
    assert eq(rd("MU2D").reshape(ng, 2), o["mu"]), "mu2d"
    assert eq(rd("DEPTH"), o["depth"]), "depth"
    assert eq(rd("CONIC_OPACITY").reshape(ng, 4), o["conic_o"]), "conic_opacity"
    # H5 on non-culled Gaussians
    live = o["touched"] > 0
    Lo = rd("RADIANCE").reshape(ng, 4)[:, :3].astype(np.float64)
    col = rd("COLOR").reshape(ng, 4)[:, :3].astype(np.float64)
    if live.any():
        dL = np.abs(Lo[live] - o["L_o"][live]) / np.maximum(1.0, np.abs(o["L_o"][live]))
        dc = np.abs(col[live] - o["color"][live])
        rep["radiance_max"], rep["color_max"], rep["color_mean"] = dL.max(), dc.max(), dc.mean()
        assert dL.max() <= IMG_MAX, "radiance max %g" % dL.max()
        assert dc.max() <= IMG_MAX and dc.mean() <= IMG_MEAN, "colour max %g mean %g" % (dc.max(), dc.mean())
    # H7-H9 (bit-exact)
    D = int(rd("NUM_DUPLICATES")[0])
    assert D == len(o["keys"]), "D %d vs %d" % (D, len(o["keys"]))
    assert eq(rd("KEYS_SORTED"), o["keys"]), "sorted keys"
    assert eq(rd("VALS_SORTED"), o["vals"]), "sorted vals"
    assert eq(rd("TILE_RANGES").reshape(-1, 2), o["ranges"]), "tile ranges"
    # H10.  Unflagged pixels: north_star bounds on image and T_final, n_contrib exact.  Flagged pixels (A38: one
    # of the blend's threshold decisions is within fp32 reach of flipping; ~1e-5 of the pixels): one alpha ~ 1/255
    # contribution may flip, so image and T_final are held to 1/255 + 2e-3 there and n_contrib is not constrained.
    d = np.abs(img.astype(np.float64) - o["image"]).max(-1)
    fl = o["flags"].astype(bool)
    rep["image_max"], rep["image_mean"], rep["flagged"] = d[~fl].max() if (~fl).any() else 0.0, d.mean(), int(fl.sum())
    # how many pixels may be flagged: 1e-4 of them on the configs; the band has a fixed RELATIVE width (A38), so the count really
    # scales with the blended (pixel, entry) pairs -- the randomised sweep (large Gaussians seen close up) bounds it per pair
    pairs = float(o["n_contrib"].astype(np.int64).sum())
    # (a count of rare events: three standard deviations of a Poisson count on top of the rate -- sweep seed 56494 has 3 flagged
    # pixels where the rate alone allows 2.6)
    lam = flag_per_pair * pairs if flag_per_pair is not None else 0.0
    allowed = max(2.0, 1e-4 * fl.size) if flag_per_pair is None else max(2.0, lam + 3.0 * np.sqrt(lam))
    assert fl.sum() <= allowed, "flag band too wide: %d px (allowed %.0f)" % (fl.sum(), allowed)
    assert rep["image_max"] <= IMG_MAX, "image max %g" % rep["image_max"]
    assert d.mean() <= IMG_MEAN, "image mean %g" % d.mean()
    H, W = img.shape[:2]
    T = rd("T_FINAL").reshape(H, W).astype(np.float64)
    dT = np.abs(T - o["T_final"])
    if fl.any():
        # what a flipped decision can move (A38): alpha against 1/255 -- one contribution of 1/255; the stopping rule -- the entry
        # that takes T to 1e-4 weighs alpha T = 1e-4 alpha / (1 - alpha) <= 9.9e-3 (sweep seed 109469: 7.7e-3); the sign of power
        # -- a whole contribution (not bounded)
        kind = o["flags"].astype(np.int64)
        bound = IMG_MAX + np.where(kind & 1, 1.0 / 255.0, 0.0) + np.where(kind & 2, 9.9e-3, 0.0) + np.where(kind & 4, 1.0, 0.0)
        assert (d[fl] <= bound[fl]).all(), "flagged pixels: image off by %g" % (d[fl] - bound[fl]).max()
        assert (dT[fl] <= bound[fl]).all(), "flagged pixels: T_final off by %g" % (dT[fl] - bound[fl]).max()
    assert dT[~fl].max() <= IMG_MAX, "T_final"
    nc = rd("N_CONTRIB").reshape(H, W)
    rep["n_contrib_mismatch"] = int((nc != o["n_contrib"])[~fl].sum())
    assert rep["n_contrib_mismatch"] == 0, "n_contrib differs on %d unflagged pixels" % rep["n_contrib_mismatch"]
    return rep
