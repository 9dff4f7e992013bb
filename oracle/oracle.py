"""ctypes front-end of the CPU oracle (oracle/rga_oracle.cpp).  TEST INFRASTRUCTURE ONLY: imported by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs; never by the product package.

`avatar_load(inputs)` mirrors step L0 and `render_frame(av, inputs, ...)` runs H1..H10 in the paper's order
(Fig.1 :84, test-time flow :197) and returns every intermediate as numpy arrays.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_emit_sort.restype = C.c_int64
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def set_threads(n):
    os.environ["OMP_NUM_THREADS"] = str(n)


# ------------------------------------------------------------------------------------------------ steps
def knn(q, v, K):
    q, v = _f32(q), _f32(v)
    idx = np.empty((len(q), K), np.int32); d2 = np.empty((len(q), K), np.float32)
    lib().orc_knn(_p(q), C.c_int(len(q)), _p(v), C.c_int(len(v)), C.c_int(K), _p(idx), _p(d2))
    return idx, d2


def interp_weights(d2):
    d2 = _f32(d2); out = np.empty_like(d2)
    lib().orc_interp_weights(_p(d2), C.c_int(d2.shape[0]), C.c_int(d2.shape[1]), _p(out))
    return out


def interp_attr(idx, ubar, attr):
    attr = _f32(attr)
    a2 = attr.reshape(len(attr), -1)
    out = np.empty((len(idx), a2.shape[1]), np.float32)
    lib().orc_interp_attr(_p(idx), _p(ubar), C.c_int(len(idx)), C.c_int(idx.shape[1]), _p(a2), C.c_int(a2.shape[1]), _p(out))
    return out.reshape((len(idx),) + attr.shape[1:])


def interp_quat(idx, ubar, vq):
    vq = _f32(vq); out = np.empty((len(idx), 4), np.float32)
    lib().orc_interp_quat(_p(idx), _p(ubar), C.c_int(len(idx)), C.c_int(idx.shape[1]), _p(vq), _p(out))
    return out


def normalize_rows3(v):
    v = _f32(v).copy()
    lib().orc_normalize_rows3(_p(v), C.c_int(len(v)))
    return v


def vertex_normals(x, faces):
    """Area-weighted vertex normals of the canonical mesh (reading A40): what `vert_normal = None` means."""
    x = _f32(x); faces = np.ascontiguousarray(faces, np.int32)
    out = np.empty_like(x)
    lib().orc_vertex_normals(_p(x), _p(faces), C.c_int(len(x)), C.c_int(len(faces)), _p(out))
    return out


def skin(x, dx, n, w, G):
    x, n, w, G = _f32(x), _f32(n), _f32(w), _f32(G)
    dx = None if dx is None else _f32(dx)
    xo = np.empty_like(x); no = np.empty_like(x); M = np.empty((len(x), 12), np.float32)
    lib().orc_skin(_p(x), _p(dx), _p(n), _p(w), C.c_int(len(x)), C.c_int(w.shape[1]), _p(G), _p(xo), _p(no), _p(M))
    return xo, no, M


def gauss_cov(M, q, s):
    M, q, s = _f32(M), _f32(q), _f32(s)
    out = np.empty((len(q), 6), np.float32)
    lib().orc_gauss_cov(_p(M), _p(q), _p(s), C.c_int(len(q)), _p(out))
    return out


def window(x):
    x = _f32(x); c = np.empty(3, np.float32); r = C.c_float(0)
    lib().orc_window(_p(x), C.c_int(len(x)), _p(c), C.byref(r))
    return c, np.float32(r.value)


def light_frames(dirs):
    dirs = _f32(dirs); out = np.empty((len(dirs), 9), np.float32)
    lib().orc_light_frames(_p(dirs), C.c_int(len(dirs)), _p(out))
    return out


def vis_raster(xp, faces, dirs, R, c, r, want_ids=True, cull=False):
    xp, dirs, c = _f32(xp), _f32(dirs), _f32(c)
    faces = np.ascontiguousarray(faces, np.int32)
    K = len(dirs)
    z = np.empty((K, R, R), np.uint32)
    ids = np.empty((K, R, R), np.int32) if want_ids else None
    lib().orc_vis_raster(_p(xp), C.c_int(len(xp)), _p(faces), C.c_int(len(faces)), _p(dirs), C.c_int(K), C.c_int(R),
                         _p(c), C.c_float(r), _p(z), _p(ids), C.c_int(int(cull)))
    return z, ids


def vis_depth_test(xg, ng, dirs, R, c, r, zmap, bias_texels, bias_world, slope_max):
    xg, ng, dirs, c = _f32(xg), _f32(ng), _f32(dirs), _f32(c)
    K = len(dirs)
    bits = np.empty((len(xg), (K + 31) // 32), np.uint32)
    lib().orc_vis_depth_test(_p(xg), _p(ng), C.c_int(len(xg)), _p(dirs), C.c_int(K), C.c_int(R), _p(c), C.c_float(r),
                             _p(zmap), C.c_float(bias_texels), C.c_float(bias_world), C.c_float(slope_max), _p(bits))
    return bits


def vis_paper(idmap, faces, nv, knn_v, want_stages=False):
    K, R = idmap.shape[0], idmap.shape[1]
    faces = np.ascontiguousarray(faces, np.int32)
    vcount = np.empty((nv, K), np.uint8)
    st = [np.empty((K, nv), np.uint8) for _ in range(3)] if want_stages else [None] * 3
    lib().orc_vis_paper(_p(idmap), _p(faces), C.c_int(len(faces)), C.c_int(nv), C.c_int(K), C.c_int(R), _p(knn_v),
                        C.c_int(knn_v.shape[1]), _p(vcount), _p(st[0]), _p(st[1]), _p(st[2]))
    return (vcount, st) if want_stages else vcount


def vis_gauss(vcount, knn_g, ubar, Kv):
    knn_g = np.ascontiguousarray(knn_g, np.int32); ubar = _f32(ubar)
    ng, K = len(knn_g), vcount.shape[1]
    out = np.empty((ng, K), np.float64)
    lib().orc_vis_gauss(_p(vcount), _p(knn_g), _p(ubar), C.c_int(ng), C.c_int(knn_g.shape[1]), C.c_int(K), C.c_int(Kv), _p(out))
    return out


def env_table(rows, cols):
    w = np.empty((rows * cols, 3), np.float64); A = np.empty(rows * cols, np.float64)
    lib().orc_env_table(C.c_int(rows), C.c_int(cols), _p(w), _p(A))
    return w, A


def brdf(wi, wo, n, albedo, rough, spec):
    a = [np.ascontiguousarray(v, np.float64) for v in (wi, wo, n, albedo)]
    out = np.empty(3, np.float64)
    lib().orc_brdf(_p(a[0]), _p(a[1]), _p(a[2]), _p(a[3]), C.c_double(rough), C.c_double(spec), _p(out))
    return out


def shade(xg, ng, alb, rough, spec, cam_pos, env, t2d, vis_mode, bits=None, vg=None, K=0, gamma=2.2):
    xg, ng, alb, rough, spec, cam_pos, env = map(_f32, (xg, ng, alb, rough, spec, cam_pos, env))
    rows, cols = env.shape[0], env.shape[1]
    n = len(xg)
    Lo = np.empty((n, 3), np.float64); cg = np.empty((n, 3), np.float64)
    t2d = None if t2d is None else np.ascontiguousarray(t2d, np.int32)
    lib().orc_shade(_p(xg), _p(ng), _p(alb), _p(rough), _p(spec), C.c_int(n), _p(cam_pos), _p(env), C.c_int(rows),
                    C.c_int(cols), _p(t2d), C.c_int(vis_mode), _p(bits), _p(vg), C.c_int(K), C.c_double(gamma), _p(Lo), _p(cg))
    return Lo, cg


def camera_array(cam):
    return np.concatenate([_f32(cam["R_wc"]).reshape(9), _f32(cam["t_wc"]).reshape(3),
                           np.array([cam["fx"], cam["fy"], cam["cx"], cam["cy"], cam["width"], cam["height"],
                                     cam["z_near"]], np.float32)]).astype(np.float32)


def project(xg, ng, cov6, opac, cam):
    xg, ng, cov6 = _f32(xg), _f32(ng), _f32(cov6)
    opac = None if opac is None else _f32(opac)
    n = len(xg); ca = camera_array(cam)
    o = dict(mu=np.empty((n, 2), np.float32), depth=np.empty(n, np.float32), conic_o=np.empty((n, 4), np.float32),
             rect=np.empty((n, 4), np.int32), touched=np.empty(n, np.uint32), radius=np.empty(n, np.int32))
    lib().orc_project(_p(xg), _p(ng), _p(cov6), _p(opac), C.c_int(n), _p(ca), _p(o["mu"]), _p(o["depth"]),
                      _p(o["conic_o"]), _p(o["rect"]), _p(o["touched"]), _p(o["radius"]))
    return o


def emit_sort(depth, rect, touched, TX):
    D = int(touched.astype(np.int64).sum())
    keys = np.empty(max(D, 1), np.uint64); vals = np.empty(max(D, 1), np.uint32)
    d = lib().orc_emit_sort(_p(depth), _p(rect), _p(touched), C.c_int(len(depth)), C.c_int(TX), _p(keys), _p(vals))
    assert d == D
    return keys[:D], vals[:D]


def tile_ranges(keys, ntiles):
    r = np.zeros((ntiles, 2), np.uint32)
    k = np.ascontiguousarray(keys, np.uint64)
    lib().orc_tile_ranges(_p(k), C.c_int64(len(k)), C.c_int(ntiles), _p(r))
    return r


def composite(vals, ranges, mu, conic_o, col, bg, W, H):
    col = np.ascontiguousarray(col, np.float64); bg = _f32(bg)
    vals = np.ascontiguousarray(vals, np.uint32)
    if len(vals) == 0:
        vals = np.zeros(1, np.uint32)
    img = np.empty((H, W, 3), np.float64); T = np.empty((H, W), np.float64)
    nc = np.empty((H, W), np.uint32); fl = np.empty((H, W), np.uint8)
    lib().orc_composite(_p(vals), _p(ranges), _p(mu), _p(conic_o), _p(col), _p(bg), C.c_int(W), C.c_int(H), _p(img),
                        _p(T), _p(nc), _p(fl))
    return img, T, nc, fl


def composite_bruteforce(depth, rect, touched, mu, conic_o, col, bg, W, H):
    col = np.ascontiguousarray(col, np.float64); bg = _f32(bg)
    img = np.empty((H, W, 3), np.float64); T = np.empty((H, W), np.float64); nc = np.empty((H, W), np.uint32)
    lib().orc_composite_bruteforce(_p(depth), _p(rect), _p(touched), C.c_int(len(depth)), _p(mu), _p(conic_o), _p(col),
                                   _p(bg), C.c_int(W), C.c_int(H), _p(img), _p(T), _p(nc))
    return img, T, nc


# ------------------------------------------------------------------------------------------------ pipeline
K_G, K_V = 3, 19


def disp_mlp(x, theta, m):
    """Displacement network d(x, theta) (readings A26-A28), fp64, plain matrix products:
    h0 = [sin(2 pi B x), cos(2 pi B x), theta]; h_l = relu(W_l h_{l-1} + b_l) for the hidden layers; dx = W_o h + b_o.
    m: dict with rff [F,3], W1 [width, 2F+P], b1, Wh [L-1, width, width], bh [L-1, width], Wo [3, width], bo [3]."""
    x = np.asarray(x, np.float64); theta = np.asarray(theta, np.float64)
    p = 2.0 * np.pi * (x @ np.asarray(m["rff"], np.float64).T)
    h = np.concatenate([np.sin(p), np.cos(p), np.broadcast_to(theta, (len(x), len(theta)))], axis=1)
    h = np.maximum(h @ np.asarray(m["W1"], np.float64).T + np.asarray(m["b1"], np.float64), 0.0)
    for W, b in zip(np.asarray(m["Wh"], np.float64), np.asarray(m["bh"], np.float64)):
        h = np.maximum(h @ W.T + b, 0.0)
    return h @ np.asarray(m["Wo"], np.float64).T + np.asarray(m["bo"], np.float64)


def densify_density(knn_g, faces, vert_pos, d0, p0, rnd):
    """Algorithm 1, "Gaussian densification based on density" (text :475-479 and :173), step by step
    in the paper's order and names.  knn_g: S_g [N_g, K_g]; faces [N_f, 3]; vert_pos [N_v, 3] canonical x; rnd: uint32
    [3 * n] raw random numbers drawn by the caller (one for the multinomial draw, two for the placement of each added
    Gaussian); at most len(rnd) // 3 Gaussians are produced.
    Readings (A29-A31): d_f and P are fp32; the multinomial sample is n draws by inverse CDF over P held in
    fixed point (P * 2^16 rounded to nearest), so that sums are exact integers: N' = floor(sum(P) * p0), draw j picks the
    first triangle whose running sum exceeds floor(rnd[3j] / 2^32 * sum); "randomly add on the triangle" = the uniform
    barycentric map (1 - sqrt(r1), sqrt(r1)(1 - r2), sqrt(r1) r2) with r = (rnd >> 8) / 2^24.
    Returns dict: D_v int32 [N_v], P_fix uint32 [N_f], n_add (N'), tri int32 [n], n_g int32 [N_f] (histogram of tri),
    pos float32 [n, 3]."""
    knn_g = np.asarray(knn_g); faces = np.asarray(faces); x = _f32(vert_pos)
    rnd = np.asarray(rnd, dtype=np.uint32)
    N_v, N_f, K_g = len(x), len(faces), knn_g.shape[1]
    # "for Gaussian index i: for vertex index k in S_g^i: D_v[k] += 1"
    D_v = np.zeros(N_v, np.int64)
    np.add.at(D_v, knn_g.reshape(-1), 1)
    # "for triangle index i: for vertex index k in f^i: d_f[i] += D_v[k];  d_f[i] /= (6 x K_g)"
    d_f = np.zeros(N_f, np.float32)
    for c in range(3):
        d_f = d_f + D_v[faces[:, c]].astype(np.float32)            # integers < 2^24: exact in fp32
    d_f = d_f / np.float32(6 * K_g)
    # "P = max(0, d_0 - d_f)"
    P = np.maximum(np.float32(0.0), np.float32(d0) - d_f)
    P_fix = np.rint(P.astype(np.float64) * 65536.0).astype(np.uint64)
    total = int(P_fix.sum())
    # "N_g' = sum(P) x p_0"
    n_add = int(np.floor(float(total) * float(np.float32(p0)) / 65536.0))
    n = min(n_add, len(rnd) // 3)
    # "n_g = MultinomialSample(P / sum(P), N_g')"
    cdf = np.cumsum(P_fix)
    tri = np.empty(n, np.int32)
    for j in range(n):
        target = (int(rnd[3 * j]) * total) >> 32
        tri[j] = int(np.searchsorted(cdf, np.uint64(target), side="right"))
    n_g = np.bincount(tri, minlength=N_f).astype(np.int32)
    # "randomly add n_g[i] Gaussians on the i-th triangle"
    r1 = (rnd[1:3 * n:3] >> np.uint32(8)).astype(np.float32) * np.float32(2.0 ** -24)
    r2 = (rnd[2:3 * n:3] >> np.uint32(8)).astype(np.float32) * np.float32(2.0 ** -24)
    sq = np.sqrt(r1)
    b0 = np.float32(1.0) - sq; b1 = sq * (np.float32(1.0) - r2); b2 = sq * r2
    f = faces[tri]
    pos = (b0[:, None] * x[f[:, 0]] + b1[:, None] * x[f[:, 1]]) + b2[:, None] * x[f[:, 2]]
    return {"D_v": D_v.astype(np.int32), "P_fix": P_fix.astype(np.uint32), "n_add": n_add, "tri": tri, "n_g": n_g,
            "pos": pos.astype(np.float32)}


def avatar_load(inp):
    """L0: KNN sets S_g, S_v and Eq.1 interpolation of the pose-independent attributes."""
    av = {}
    av["knn_g"], d2g = knn(inp["gauss_pos"], inp["vert_pos"], K_G)
    av["ubar_g"] = interp_weights(d2g)
    kv = min(K_V, len(inp["vert_pos"]))
    av["knn_v"], _ = knn(inp["vert_pos"], inp["vert_pos"], kv)
    i, u = av["knn_g"], av["ubar_g"]
    av["vert_normal"] = _f32(inp["vert_normal"]) if inp.get("vert_normal") is not None else vertex_normals(inp["vert_pos"], inp["faces"])
    av["normal_g"] = normalize_rows3(interp_attr(i, u, av["vert_normal"]))
    av["albedo_g"] = interp_attr(i, u, inp["vert_albedo"])
    av["rough_g"] = interp_attr(i, u, inp["vert_rough"])
    av["spec_g"] = interp_attr(i, u, inp["vert_spec"])
    av["skin_w_g"] = interp_attr(i, u, inp["vert_skin_w"])
    av["disp_g"] = interp_attr(i, u, inp["vert_disp"])
    # the paper's layout: rotation and scale as vertex attributes, used when no per-Gaussian array is given
    if inp.get("gauss_quat") is None and inp.get("vert_quat") is not None:
        av["quat_g"] = interp_quat(i, u, inp["vert_quat"])
    if inp.get("gauss_scale") is None and inp.get("vert_scale") is not None:
        av["scale_g"] = interp_attr(i, u, inp["vert_scale"])
    return av


def render_frame(av, inp, frame=0, vis_mode=0, camera=None, stop_after=None, gauss_chunk=None, timings=None):
    """H1..H10.  vis_mode 0 = depth test (north_star), 1 = paper (Eq.3-4), 2 = no visibility (v = 1).
    gauss_chunk (paper mode only): evaluate Eq.1-of-v and the shading in chunks of that many Gaussians, so that the
    [N_g, K] double table of v_g is never held whole (8 GB at config 4); the arithmetic per Gaussian is unchanged and
    o["vis_g"] is then not returned.
    timings: optional dict; the wall-clock seconds of each stage (skin, visibility, shade, splat) are added to it
    (bench.py's cpu_baseline leg)."""
    import time as _time
    t_prev = [_time.perf_counter()]

    def lap(name):
        if timings is not None:
            now = _time.perf_counter()
            timings[name] = timings.get(name, 0.0) + (now - t_prev[0])
            t_prev[0] = now
    o = {}
    G = inp["bone_mats"][frame]
    o["vert_posed"], o["vert_normal_posed"], _ = skin(inp["vert_pos"], inp["vert_disp"], av["vert_normal"],
                                                      inp["vert_skin_w"], G)
    o["gauss_posed"], o["gauss_normal_posed"], M = skin(inp["gauss_pos"], av["disp_g"], av["normal_g"], av["skin_w_g"], G)
    o["cov6"] = gauss_cov(M, av["quat_g"] if "quat_g" in av else inp["gauss_quat"], av["scale_g"] if "scale_g" in av else inp["gauss_scale"])
    o["win_c"], o["win_r"] = window(o["vert_posed"])
    lap("skin")
    if stop_after == "skin":
        return o
    dirs, R = inp["vis_dirs"], inp["vis_res"]
    K = len(dirs)
    bits = vg = None
    if vis_mode in (0, 1):
        o["zmap"], o["idmap"] = vis_raster(o["vert_posed"], inp["faces"], dirs, R, o["win_c"], o["win_r"], want_ids=True,
                                           cull=bool(inp.get("vis_cull_backfaces", False)))
        lap("vis_raster")
    if vis_mode == 0:
        bits = o["visbits"] = vis_depth_test(o["gauss_posed"], o["gauss_normal_posed"], dirs, R, o["win_c"], o["win_r"],
                                             o["zmap"], inp["depth_bias_texels"], inp["depth_bias_world"], inp["slope_max"])
        lap("vis_depth_test")
    elif vis_mode == 1:
        o["vcount"] = vis_paper(o["idmap"], inp["faces"], len(inp["vert_pos"]), av["knn_v"])
        if not gauss_chunk:
            vg = o["vis_g"] = vis_gauss(o["vcount"], av["knn_g"], av["ubar_g"], av["knn_v"].shape[1])
        lap("vis_paper")
    if stop_after == "vis":
        return o
    env = inp["env"][inp["env_of_frame"][frame]]
    if vis_mode == 1 and gauss_chunk:
        ng = len(o["gauss_posed"])
        o["L_o"] = np.empty((ng, 3), np.float64); o["color"] = np.empty((ng, 3), np.float64)
        for a in range(0, ng, gauss_chunk):
            b = min(ng, a + gauss_chunk)
            vgc = vis_gauss(o["vcount"], av["knn_g"][a:b], av["ubar_g"][a:b], av["knn_v"].shape[1])
            o["L_o"][a:b], o["color"][a:b] = shade(o["gauss_posed"][a:b], o["gauss_normal_posed"][a:b], av["albedo_g"][a:b],
                                                   av["rough_g"][a:b], av["spec_g"][a:b], inp["cam_pos"], env, inp["texel_to_dir"],
                                                   1, None, vgc, K, inp["gamma"])
    else:
        o["L_o"], o["color"] = shade(o["gauss_posed"], o["gauss_normal_posed"], av["albedo_g"], av["rough_g"], av["spec_g"],
                                     inp["cam_pos"], env, inp["texel_to_dir"], vis_mode, bits, vg, K, inp["gamma"])
    lap("shade")
    if stop_after == "shade":
        return o
    cam = camera or inp["camera"]
    W, H = cam["width"], cam["height"]
    TX, TY = (W + 15) // 16, (H + 15) // 16
    o.update(project(o["gauss_posed"], o["gauss_normal_posed"], o["cov6"], inp["gauss_opacity"], cam))
    o["keys"], o["vals"] = emit_sort(o["depth"], o["rect"], o["touched"], TX)
    o["ranges"] = tile_ranges(o["keys"], TX * TY)
    lap("project_sort")
    o["image"], o["T_final"], o["n_contrib"], o["flags"] = composite(o["vals"], o["ranges"], o["mu"], o["conic_o"],
                                                                     o["color"], inp["bg"], W, H)
    lap("composite")
    return o


def set_num_threads(n):
    """OpenMP thread count of the oracle library from here on (bench.py times it single-threaded and on all cores)."""
    g = C.CDLL("libgomp.so.1")
    g.omp_set_num_threads(C.c_int(int(n)))
