"""GPU parity of splat_backward against the fp64 autograd oracle (oracle/backward.py) on the same
seeded inputs and the same seeded dL/dimage."""
import numpy as np
import pytest

from synth import workloads

pytestmark = pytest.mark.gpu

# tolerances, as fractions of the largest reference magnitude of each gradient array ("backward"):
# fp32 sums of up to ~10^3 terms with T recovered by repeated division, ex2.approx alphas, forward colours within 2e-3
TOL_MAX, TOL_MEAN = 1e-4, 1e-6          # measured: <= 5.1e-6 and <= 2.6e-8 on configs 0 and 1


def _run(cfg, n_gauss=None, vis_mode=0, use_visibility=True, bg=None):
    import torch
    from oracle import backward as bwd
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    from parity_util import run_gpu
    inp = workloads.make(cfg, n_gauss=n_gauss)
    if bg is not None:
        inp["bg"] = np.asarray(bg, np.float32)
    cam = inp["camera"]; W, H = cam["width"], cam["height"]
    orc_av = orc.avatar_load(inp)
    o = orc.render_frame(orc_av, inp, vis_mode=vis_mode if use_visibility else 2)
    G = workloads.make_image_cotangent(cfg, W, H)
    ref = bwd.splat_backward(o["gauss_posed"], o["cov6"], o["color"], inp["gauss_opacity"], cam, inp["bg"], o["vals"], o["ranges"],
                             o["touched"], G, mu32=o["mu"], conic32=o["conic_o"])
    av, img = run_gpu(inp, vis_mode=vis_mode, use_visibility=use_visibility, keep_maps=False)
    N = len(inp["gauss_pos"])
    dev = "cuda"
    d_col = torch.full((N, 3), float("nan"), device=dev); d_op = torch.full((N,), float("nan"), device=dev)
    d_x = torch.full((N, 3), float("nan"), device=dev); d_cov = torch.full((N, 6), float("nan"), device=dev)
    rga.splat_backward(av.h, cam, inp["bg"], torch.as_tensor(np.ascontiguousarray(img, np.float32)).to(dev), torch.as_tensor(G).to(dev), d_col, d_op, d_x, d_cov)
    rga.rga_check(av.h)
    sg = av.read("SPLAT_GRAD").reshape(N, 12)
    got = {"d_col": d_col.cpu().numpy(), "d_opac": d_op.cpu().numpy(), "d_mu": sg[:, 4:6], "d_conic": sg[:, 6:9],
           "d_x": d_x.cpu().numpy(), "d_cov6": d_cov.cpu().numpy()}
    assert np.array_equal(sg[:, 0:3], got["d_col"]) and np.array_equal(sg[:, 3], got["d_opac"])
    rep = {}
    for k, g in got.items():
        r = ref[k]
        assert np.isfinite(g).all(), k
        scale = np.abs(r).max()
        rep[k] = (float(np.abs(g - r).max() / scale), float(np.abs(g - r).mean() / scale), float(scale))
    culled = o["touched"] == 0
    for k, g in got.items():
        assert not g[culled].any(), k                                     # rows of culled Gaussians are exactly 0
    av.close()
    return rep, ref, got


@pytest.mark.parametrize("cfg,use_vis,bg", [(0, True, None), (0, False, (0.3, 0.6, 0.2)), (1, False, None), (1, False, (0.5, 0.1, 0.9))])
def test_splat_backward_matches_autograd_oracle(cfg, use_vis, bg):
    rep, ref, got = _run(cfg, use_visibility=use_vis, bg=bg)
    print(rep)
    for k, (emax, emean, scale) in rep.items():
        assert scale > 0, k
        assert emax < TOL_MAX and emean < TOL_MEAN, (k, emax, emean, scale)


def test_splat_backward_argument_checks():
    import torch
    from paper_2407_10707_b200 import binding as rga
    inp = workloads.make(0)
    cam = inp["camera"]; W, H = cam["width"], cam["height"]
    av = rga.Avatar(inp, max_width=W, max_height=H, max_vis_dirs=16, max_vis_res=32, max_env_texels=512)
    G = torch.zeros((H, W, 3), device="cuda")
    with pytest.raises(RuntimeError):
        rga.splat_backward(av.h, cam, inp["bg"], G, G)                   # nothing rendered yet
    # an attribute map overwrites the blend state of the shaded frame: its backward is refused until the frame is splatted again
    rga.pose_skin(av.h, torch.as_tensor(inp["bone_mats"][0]).cuda())
    rga.shade_gaussians(av.h, torch.as_tensor(inp["env"][0]).cuda(), inp["cam_pos"], None, inp["gamma"], False)
    img = torch.zeros((H, W, 3), device="cuda")
    rga.splat_render(av.h, cam, inp["bg"], img)
    rga.splat_backward(av.h, cam, inp["bg"], img, G)
    rga.splat_attribute(av.h, cam, inp["bg"], rga.RGA_ATTR_ALBEDO, img)
    with pytest.raises(RuntimeError):
        rga.splat_backward(av.h, cam, inp["bg"], img, G)
    rga.splat_render(av.h, cam, inp["bg"], img)
    rga.splat_backward(av.h, cam, inp["bg"], img, G)
    rga.rga_check(av.h)
    av.close()


# shading backward: the gradients scale with (1/gamma) L_o^(1/gamma - 1), i.e. they are largest for the darkest lit
# Gaussians, whose fp32 forward radiance carries the largest relative error; tolerances as fractions of the largest
# reference magnitude of each array (measured values in DESIGN.md)
SH_TOL_MAX, SH_TOL_MEAN = 2e-3, 5e-6          # measured: <= 7.5e-4 (d_x) and <= 9e-7


@pytest.mark.parametrize("cfg,vis_mode,use_vis", [(0, 0, True), (0, 1, True), (0, 0, False), (1, 0, True), (1, 1, True)])
def test_shade_backward_matches_autograd_oracle(cfg, vis_mode, use_vis):
    import torch
    from oracle import backward as bwd
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    from parity_util import run_gpu
    inp = workloads.make(cfg, n_gauss=30_000 if cfg == 1 else None)
    orc_av = orc.avatar_load(inp)
    mode = vis_mode if use_vis else 2
    o = orc.render_frame(orc_av, inp, vis_mode=mode, stop_after="shade")
    env = inp["env"][inp["env_of_frame"][0]]
    N = len(inp["gauss_pos"]); ne = env.shape[0] * env.shape[1]
    v = bwd.texel_visibility(N, ne, inp["texel_to_dir"], mode, bits=o.get("visbits"), vg=o.get("vis_g"))
    d_col = workloads.make_color_cotangent(cfg, N)
    ref = bwd.shade_backward(o["gauss_posed"], o["gauss_normal_posed"], orc_av["albedo_g"], orc_av["rough_g"], orc_av["spec_g"], inp["cam_pos"],
                             env, v, inp["gamma"], d_col)
    av, img = run_gpu(inp, vis_mode=vis_mode, use_visibility=use_vis, keep_maps=False)
    dev = "cuda"
    nanf = lambda *s: torch.full(s, float("nan"), device=dev)
    outs = dict(out_dalbedo=nanf(N, 3), out_drough=nanf(N), out_dspec=nanf(N), out_dnormal=nanf(N, 3), out_dpos=nanf(N, 3),
                out_denv=nanf(env.shape[0], env.shape[1], 3))
    rga.shade_backward(av.h, torch.as_tensor(env).to(dev), inp["cam_pos"], torch.as_tensor(d_col).to(dev),
                       texel_to_dir=torch.as_tensor(inp["texel_to_dir"]).to(dev), gamma=inp["gamma"], use_visibility=use_vis, **outs)
    rga.rga_check(av.h)
    # the library skips Gaussians that face away from the camera (their colour is never splatted); the
    # oracle's shade function does not know the camera's cull, so compare the Gaussians the forward pass keeps
    facing = ((inp["cam_pos"][None, :] - o["gauss_posed"]) * o["gauss_normal_posed"]).sum(1) >= 1e-3
    keep = facing
    rep = {}
    for name, key in (("d_alb", "out_dalbedo"), ("d_rough", "out_drough"), ("d_spec", "out_dspec"), ("d_n", "out_dnormal"), ("d_x", "out_dpos")):
        g = outs[key].cpu().numpy(); r = ref[name]
        assert np.isfinite(g).all(), name
        scale = np.abs(r[keep]).max()
        rep[name] = (float(np.abs(g[keep] - r[keep]).max() / scale), float(np.abs(g[keep] - r[keep]).mean() / scale), float(scale))
    # environment gradient: sums over all Gaussians, so the oracle's is recomputed over the kept ones only
    ref_env = bwd.shade_backward(o["gauss_posed"][keep], o["gauss_normal_posed"][keep], orc_av["albedo_g"][keep], orc_av["rough_g"][keep],
                                 orc_av["spec_g"][keep], inp["cam_pos"], env, v[keep], inp["gamma"], d_col[keep])["d_env"]
    # ... and the library's over exactly those: zero the cotangent of the others
    d_col2 = d_col.copy(); d_col2[~keep] = 0.0
    rga.shade_backward(av.h, torch.as_tensor(env).to(dev), inp["cam_pos"], torch.as_tensor(d_col2).to(dev),
                       texel_to_dir=torch.as_tensor(inp["texel_to_dir"]).to(dev), gamma=inp["gamma"], use_visibility=use_vis, out_denv=outs["out_denv"])
    ge = outs["out_denv"].cpu().numpy()
    scale = np.abs(ref_env).max()
    rep["d_env"] = (float(np.abs(ge - ref_env).max() / scale), float(np.abs(ge - ref_env).mean() / scale), float(scale))
    print(rep)
    for k, (emax, emean, scale) in rep.items():
        assert scale > 0, k
        assert emax < SH_TOL_MAX and emean < SH_TOL_MEAN, (k, emax, emean, scale)
    av.close()


@pytest.mark.parametrize("W,H,lam", [(64, 64, 0.2), (70, 45, 0.2), (512, 512, 0.2), (512, 512, 0.0), (33, 17, 1.0)])
def test_image_loss_matches_oracle(W, H, lam):
    # Eq.5: loss value and dL/dimage; fp32 window sums of 121 taps against fp64 -> 1e-5 relative on the loss, 2e-4 of the
    # largest gradient entry (sigma^2 = w*I^2 - mu^2 cancels in fp32 where the window is flat)
    import torch
    from oracle import backward as bwd
    from paper_2407_10707_b200 import binding as rga
    inp = workloads.make(0)
    av = rga.Avatar(inp, max_width=512, max_height=512, max_vis_dirs=16, max_vis_res=32, max_env_texels=512)
    img, tgt = workloads.make_image_pair(W + H, W, H)
    ref = bwd.image_loss(img, tgt, lam)
    out = torch.full((3,), float("nan"), device="cuda"); dI = torch.full((H, W, 3), float("nan"), device="cuda")
    rga.image_loss(av.h, torch.as_tensor(img).cuda(), torch.as_tensor(tgt).cuda(), lam, out, dI)
    rga.rga_check(av.h)
    got = out.cpu().numpy(); g = dI.cpu().numpy()
    assert abs(got[0] - ref["loss"]) < 1e-5 * max(ref["loss"], 1e-3), (got, ref["loss"])
    assert abs(got[1] - ref["l1"]) < 1e-6 and abs(got[2] - ref["ssim"]) < 2e-5
    scale = np.abs(ref["d_image"]).max()
    err = np.abs(g - ref["d_image"])
    print(W, H, lam, "loss", got, "grad err max/mean rel", err.max() / scale, err.mean() / scale)
    assert np.isfinite(g).all() and err.max() < 2e-4 * scale and err.mean() < 1e-5 * scale
    av.close()


@pytest.mark.parametrize("cfg,with_mlp", [(0, False), (1, False), (1, True), (2, False)])
def test_regularisers_match_oracle(cfg, with_mlp):
    # Eq.6-9: losses to 1e-5 relative (fp32 terms, double sums); Eq.6 / Eq.9 gradients are sums of +-1 / 0-1 flags: exact;
    # Eq.7 / Eq.8 gradients are sums of unit vectors: 1e-5 absolute
    import torch
    from oracle import backward as bwd
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    inp = workloads.make(cfg, n_gauss=50_000 if cfg == 2 else None)
    if cfg == 0:                                                         # a static displacement attribute, a few exactly 0
        inp["vert_disp"] = (np.random.default_rng(12).normal(0.0, 0.004, inp["vert_pos"].shape)).astype(np.float32)
        inp["vert_disp"][::7] = 0.0
    cam = inp["camera"]
    av = rga.Avatar(inp, max_width=cam["width"], max_height=cam["height"], max_vis_dirs=16, max_vis_res=32, max_env_texels=512)
    orc_av = orc.avatar_load(inp)
    disp = inp["vert_disp"]
    if with_mlp:
        mlp = workloads.make_disp_mlp(seed=2)
        rga.displacement_mlp(av.h, {k: (torch.as_tensor(v).cuda() if isinstance(v, np.ndarray) else v) for k, v in mlp.items()},
                             torch.as_tensor(mlp["theta"]).cuda())
        disp = orc.disp_mlp(inp["vert_pos"], mlp["theta"], mlp)          # fp64; the kernel's TF32 result is within 1e-2 of its scale
    ref = bwd.regularisers(inp["vert_albedo"], inp["vert_rough"], inp["vert_spec"], orc_av["knn_v"], inp["gauss_pos"], inp["vert_pos"],
                           orc_av["knn_g"], disp, inp["gauss_scale"])
    nv, ng = len(inp["vert_pos"]), len(inp["gauss_pos"])
    nanf = lambda *s: torch.full(s, float("nan"), device="cuda")
    L = nanf(4); o = dict(out_dalbedo=nanf(nv, 3), out_drough=nanf(nv), out_dspec=nanf(nv), out_dgauss_pos=nanf(ng, 3), out_ddisp=nanf(nv, 3),
                          out_dscale=nanf(ng, 3))
    rga.regularisers(av.h, 0.005, L, **o)
    rga.rga_check(av.h)
    got = L.cpu().numpy()
    print(cfg, with_mlp, got, [ref[k] for k in ("smooth", "mdist", "disp", "scale")])
    for i, k in enumerate(("smooth", "mdist", "disp", "scale")):
        tol = 2e-2 if (with_mlp and k == "disp") else 1e-5
        assert abs(got[i] - ref[k]) <= tol * abs(ref[k]) + 1e-7, (k, got[i], ref[k])
    assert np.array_equal(o["out_dalbedo"].cpu().numpy(), ref["d_albedo"]) and np.array_equal(o["out_drough"].cpu().numpy(), ref["d_rough"])
    assert np.array_equal(o["out_dspec"].cpu().numpy(), ref["d_spec"]) and np.array_equal(o["out_dscale"].cpu().numpy(), ref["d_scale"])
    assert np.abs(o["out_dgauss_pos"].cpu().numpy() - ref["d_gauss_pos"]).max() < 1e-5
    if not with_mlp:
        assert np.abs(o["out_ddisp"].cpu().numpy() - ref["d_disp"]).max() < 1e-5
    else:                                                                # unit vectors of nearly equal displacements
        assert np.abs(o["out_ddisp"].cpu().numpy() - ref["d_disp"]).max() < 5e-2
    av.close()


@pytest.mark.parametrize("cfg,n_gauss", [(0, None), (1, 100_000), (2, 50_000)])
def test_pose_backward_matches_autograd_oracle(cfg, n_gauss):
    # H2 + Eq.1 backward: every output within 1e-5 (max) / 5e-7 (mean) of its largest reference magnitude (fp32 sums; the
    # bone and vertex gradients are atomic sums over up to ~10^5 Gaussians)
    import torch
    from oracle import backward as bwd
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    inp = workloads.make(cfg, n_gauss=n_gauss)
    if cfg == 0:
        inp["vert_disp"] = (np.random.default_rng(12).normal(0.0, 0.004, inp["vert_pos"].shape)).astype(np.float32)
    cam = inp["camera"]
    av = rga.Avatar(inp, max_width=cam["width"], max_height=cam["height"], max_vis_dirs=16, max_vis_res=32, max_env_texels=512)
    orc_av = orc.avatar_load(inp)
    N, nv, B = len(inp["gauss_pos"]), len(inp["vert_pos"]), inp["bone_mats"].shape[1]
    cot = {"d_mean": workloads.make_cotangent(1, (N, 3)), "d_normal": workloads.make_cotangent(2, (N, 3)), "d_cov": workloads.make_cotangent(3, (N, 6)),
           "d_albedo": workloads.make_cotangent(4, (N, 3)), "d_rough": workloads.make_cotangent(5, (N,)), "d_spec": workloads.make_cotangent(6, (N,))}
    cot["d_normal"][::5] = 0.0                                           # some Gaussians without a normal gradient
    ref = bwd.pose_backward(inp, orc_av["knn_g"], orc_av["ubar_g"], 0, cot["d_mean"], cot["d_normal"], cot["d_cov"], cot["d_albedo"],
                            cot["d_rough"], cot["d_spec"])
    dev = "cuda"
    nanf = lambda *s: torch.full(s, float("nan"), device=dev)
    out = {"d_gauss_pos": nanf(N, 3), "d_gauss_quat": nanf(N, 4), "d_gauss_scale": nanf(N, 3), "d_bones": nanf(B, 12), "d_vert_disp": nanf(nv, 3),
           "d_vert_normal": nanf(nv, 3), "d_vert_albedo": nanf(nv, 3), "d_vert_rough": nanf(nv), "d_vert_spec": nanf(nv)}
    rga.pose_backward(av.h, torch.as_tensor(inp["bone_mats"][0]).to(dev), {k: torch.as_tensor(v).to(dev) for k, v in cot.items()}, out)
    rga.rga_check(av.h)
    rep = {}
    for k, t in out.items():
        g = t.cpu().numpy(); r = ref[k].reshape(g.shape)
        assert np.isfinite(g).all(), k
        scale = np.abs(r).max()
        rep[k] = (float(np.abs(g - r).max() / scale), float(np.abs(g - r).mean() / scale), float(scale))
    print(rep)
    for k, (emax, emean, scale) in rep.items():
        assert scale > 0 and emax < 1e-5 and emean < 5e-7, (k, emax, emean, scale)     # measured <= 8.6e-7 / 1.2e-7
    # NULL inputs are zeros: only the position path
    out2 = {"d_gauss_pos": nanf(N, 3), "d_bones": nanf(B, 12)}
    rga.pose_backward(av.h, torch.as_tensor(inp["bone_mats"][0]).to(dev), {"d_mean": torch.as_tensor(cot["d_mean"]).to(dev)}, out2)
    z3, z1, z6 = np.zeros((N, 3)), np.zeros(N), np.zeros((N, 6))
    ref2 = bwd.pose_backward(inp, orc_av["knn_g"], orc_av["ubar_g"], 0, cot["d_mean"], z3, z6, z3, z1, z1)
    assert np.abs(out2["d_bones"].cpu().numpy() - ref2["d_bones"]).max() < 1e-4 * np.abs(ref2["d_bones"]).max()
    av.close()


def test_training_backward_chain_matches_oracle_chain():
    # the whole backward of one training view at config 0: Eq.5 image loss -> splat_backward -> shade_backward ->
    # pose_backward, each stage fed by the previous one, against the same chain of oracle functions.  Catches a
    # mismatch of conventions between stages (layouts, which gradient feeds which input); per-stage accuracy is
    # tested above; tolerance 1e-3 (max) / 1e-5 (mean) of each array's largest reference magnitude.
    import torch
    from oracle import backward as bwd
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    from parity_util import run_gpu
    inp = workloads.make(0)
    cam = inp["camera"]; W, H = cam["width"], cam["height"]
    env = inp["env"][inp["env_of_frame"][0]]
    N, nv, B = len(inp["gauss_pos"]), len(inp["vert_pos"]), inp["bone_mats"].shape[1]
    _, target = workloads.make_image_pair(7, W, H)
    # ---- oracle chain
    orc_av = orc.avatar_load(inp)
    o = orc.render_frame(orc_av, inp, vis_mode=0)
    l = bwd.image_loss(o["image"], target, 0.2)
    sp = bwd.splat_backward(o["gauss_posed"], o["cov6"], o["color"], inp["gauss_opacity"], cam, inp["bg"], o["vals"], o["ranges"], o["touched"],
                            l["d_image"], mu32=o["mu"], conic32=o["conic_o"])
    v = bwd.texel_visibility(N, env.shape[0] * env.shape[1], inp["texel_to_dir"], 0, bits=o["visbits"])
    sh = bwd.shade_backward(o["gauss_posed"], o["gauss_normal_posed"], orc_av["albedo_g"], orc_av["rough_g"], orc_av["spec_g"], inp["cam_pos"],
                            env, v, inp["gamma"], sp["d_col"])
    ref = bwd.pose_backward(inp, orc_av["knn_g"], orc_av["ubar_g"], 0, sp["d_x"] + sh["d_x"], sh["d_n"], sp["d_cov6"], sh["d_alb"], sh["d_rough"],
                            sh["d_spec"])
    # ---- library chain
    dev = "cuda"
    av, img = run_gpu(inp, vis_mode=0, keep_maps=False)
    z = lambda *s: torch.zeros(s, device=dev)
    d_img = z(H, W, 3); loss = z(3)
    img_d = torch.as_tensor(np.ascontiguousarray(img, np.float32)).to(dev)
    rga.image_loss(av.h, img_d, torch.as_tensor(target).to(dev), 0.2, loss, d_img)
    d_col, d_op, d_mean, d_cov = z(N, 3), z(N), z(N, 3), z(N, 6)
    rga.splat_backward(av.h, cam, inp["bg"], img_d, d_img, d_col, d_op, d_mean, d_cov)
    s_out = dict(out_dalbedo=z(N, 3), out_drough=z(N), out_dspec=z(N), out_dnormal=z(N, 3), out_dpos=z(N, 3), out_denv=z(env.shape[0], env.shape[1], 3))
    rga.shade_backward(av.h, torch.as_tensor(env).to(dev), inp["cam_pos"], d_col, texel_to_dir=torch.as_tensor(inp["texel_to_dir"]).to(dev),
                       gamma=inp["gamma"], use_visibility=True, **s_out)
    out = {"d_gauss_pos": z(N, 3), "d_gauss_quat": z(N, 4), "d_gauss_scale": z(N, 3), "d_bones": z(B, 12), "d_vert_disp": z(nv, 3),
           "d_vert_normal": z(nv, 3), "d_vert_albedo": z(nv, 3), "d_vert_rough": z(nv), "d_vert_spec": z(nv)}
    rga.pose_backward(av.h, torch.as_tensor(inp["bone_mats"][0]).to(dev),
                      {"d_mean": d_mean, "d_mean2": s_out["out_dpos"], "d_normal": s_out["out_dnormal"], "d_cov": d_cov, "d_albedo": s_out["out_dalbedo"],
                       "d_rough": s_out["out_drough"], "d_spec": s_out["out_dspec"]}, out)
    rga.rga_check(av.h)
    assert abs(loss[0].item() - l["loss"]) < 1e-4 * l["loss"]
    rep = {}
    for k, t in list(out.items()) + [("d_env", s_out["out_denv"])]:
        g = t.cpu().numpy(); r = (sh["d_env"] if k == "d_env" else ref[k]).reshape(g.shape)
        scale = np.abs(r).max()
        rep[k] = (float(np.abs(g - r).max() / scale), float(np.abs(g - r).mean() / scale), float(scale))
    print(rep)
    for k, (emax, emean, scale) in rep.items():
        assert scale > 0 and emax < 1e-3 and emean < 1e-5, (k, emax, emean, scale)     # measured <= 4e-5 / 4.2e-7
    av.close()


def _retarget(inp, W, H):
    cam = dict(inp["camera"])
    fy = np.float32(0.5 * H / np.tan(np.deg2rad(20.0)))
    cam.update(width=W, height=H, fx=fy, fy=fy, cx=np.float32(W / 2), cy=np.float32(H / 2))
    inp["camera"] = cam


@pytest.mark.parametrize("n_gauss,W,H", [(777, 70, 50), (12_000, 16, 16), (1, 33, 17)])
def test_backward_edge_shapes(n_gauss, W, H):
    # ragged image (partial tile row and column) with a non-black background; ONE tile whose list has ~6k entries (about a
    # hundred segments fold into each pixel's prefix); a single Gaussian.  Whole chain splat -> shade -> pose.
    import torch
    from oracle import backward as bwd
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    from parity_util import run_gpu
    inp = workloads.make(0, n_gauss=n_gauss)
    inp["bg"] = np.array([0.1, 0.2, 0.3], np.float32)
    _retarget(inp, W, H)
    cam = inp["camera"]
    env = inp["env"][inp["env_of_frame"][0]]
    N, nv, B = len(inp["gauss_pos"]), len(inp["vert_pos"]), inp["bone_mats"].shape[1]
    orc_av = orc.avatar_load(inp)
    o = orc.render_frame(orc_av, inp, vis_mode=0)
    G = workloads.make_image_cotangent(n_gauss, W, H)
    sp = bwd.splat_backward(o["gauss_posed"], o["cov6"], o["color"], inp["gauss_opacity"], cam, inp["bg"], o["vals"], o["ranges"], o["touched"], G,
                            mu32=o["mu"], conic32=o["conic_o"])
    v = bwd.texel_visibility(N, env.shape[0] * env.shape[1], inp["texel_to_dir"], 0, bits=o["visbits"])
    sh = bwd.shade_backward(o["gauss_posed"], o["gauss_normal_posed"], orc_av["albedo_g"], orc_av["rough_g"], orc_av["spec_g"], inp["cam_pos"],
                            env, v, inp["gamma"], sp["d_col"])
    ref = bwd.pose_backward(inp, orc_av["knn_g"], orc_av["ubar_g"], 0, sp["d_x"] + sh["d_x"], sh["d_n"], sp["d_cov6"], sh["d_alb"], sh["d_rough"],
                            sh["d_spec"])
    dev = "cuda"
    av, img = run_gpu(inp, vis_mode=0, keep_maps=False)
    z = lambda *s: torch.zeros(s, device=dev)
    img_d = torch.as_tensor(np.ascontiguousarray(img, np.float32)).to(dev)
    d_col, d_op, d_mean, d_cov = z(N, 3), z(N), z(N, 3), z(N, 6)
    rga.splat_backward(av.h, cam, inp["bg"], img_d, torch.as_tensor(G).to(dev), d_col, d_op, d_mean, d_cov)
    s_out = dict(out_dalbedo=z(N, 3), out_drough=z(N), out_dspec=z(N), out_dnormal=z(N, 3), out_dpos=z(N, 3), out_denv=z(env.shape[0], env.shape[1], 3))
    rga.shade_backward(av.h, torch.as_tensor(env).to(dev), inp["cam_pos"], d_col, texel_to_dir=torch.as_tensor(inp["texel_to_dir"]).to(dev),
                       gamma=inp["gamma"], use_visibility=True, **s_out)
    out = {"d_gauss_pos": z(N, 3), "d_gauss_quat": z(N, 4), "d_gauss_scale": z(N, 3), "d_bones": z(B, 12), "d_vert_disp": z(nv, 3),
           "d_vert_normal": z(nv, 3), "d_vert_albedo": z(nv, 3), "d_vert_rough": z(nv), "d_vert_spec": z(nv)}
    rga.pose_backward(av.h, torch.as_tensor(inp["bone_mats"][0]).to(dev),
                      {"d_mean": d_mean, "d_mean2": s_out["out_dpos"], "d_normal": s_out["out_dnormal"], "d_cov": d_cov, "d_albedo": s_out["out_dalbedo"],
                       "d_rough": s_out["out_drough"], "d_spec": s_out["out_dspec"]}, out)
    rga.rga_check(av.h)
    pairs = [("d_col", d_col, sp["d_col"]), ("d_opac", d_op, sp["d_opac"]), ("d_x", d_mean, sp["d_x"]), ("d_cov6", d_cov, sp["d_cov6"]),
             ("d_env", s_out["out_denv"], sh["d_env"])] + [(k, t, ref[k]) for k, t in out.items()]
    rep = {}
    for k, t, r in pairs:
        g = t.cpu().numpy(); r = np.asarray(r).reshape(g.shape)
        assert np.isfinite(g).all(), k
        scale = np.abs(r).max()
        if scale == 0:                                                    # e.g. the single Gaussian faces away: everything is 0
            assert not g.any(), k
            continue
        rep[k] = (float(np.abs(g - r).max() / scale), float(np.abs(g - r).mean() / scale))
    print(n_gauss, rep)
    for k, (emax, emean) in rep.items():
        assert emax < 2e-3 and emean < 1e-4, (k, emax, emean)
    av.close()


def test_image_loss_tiny_images_and_argument_checks():
    import torch
    from oracle import backward as bwd
    from paper_2407_10707_b200 import binding as rga
    inp = workloads.make(0)
    av = rga.Avatar(inp, max_width=64, max_height=64, max_vis_dirs=16, max_vis_res=32, max_env_texels=512)
    for (W, H) in [(1, 1), (5, 3), (11, 11)]:                             # the window is wider than the image: all border
        img, tgt = workloads.make_image_pair(W * 31 + H, W, H)
        img[:] = np.clip(tgt + 0.1, 0, 1)                                # (the generator's black corner would cover a 1x1 image)
        ref = bwd.image_loss(img, tgt, 0.2)
        out = torch.zeros(3, device="cuda"); dI = torch.zeros((H, W, 3), device="cuda")
        rga.image_loss(av.h, torch.as_tensor(img).cuda(), torch.as_tensor(tgt).cuda(), 0.2, out, dI)
        rga.rga_check(av.h)
        assert abs(out[0].item() - ref["loss"]) < 1e-5 * max(ref["loss"], 1e-3)
        assert np.abs(dI.cpu().numpy() - ref["d_image"]).max() < 2e-4 * np.abs(ref["d_image"]).max()
    big = torch.zeros((65, 64, 3), device="cuda")
    with pytest.raises(RuntimeError):
        rga.image_loss(av.h, big, big, 0.2)                              # larger than the avatar's max_height
    with pytest.raises(RuntimeError):
        rga.image_loss(av.h, big[:64], big[:64], 1.5)                    # lambda outside [0, 1]
    av.close()
