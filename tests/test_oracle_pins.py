"""Pins for the CPU oracle (oracle/): each check ties one oracle function to something OTHER than itself --
a closed form, a library routine, an invariant, a brute force on tiny inputs -- so that a dropped term, wrong
sign/index or transposed operand fails here.  No GPU.  Citations are PAPER.md lines / DESIGN.md readings."""
import os

import numpy as np
import pytest

from oracle import oracle as orc
from synth import mesh as smesh
from synth import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    rows = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            rows.append([float(t) for t in line.split()])
    return np.array(rows)


# ------------------------------------------------------------------ L0: KNN + Eq.1
def test_knn_matches_kdtree_and_tie_rule():
    from scipy.spatial import cKDTree
    r = np.random.default_rng(1)
    v = r.normal(size=(500, 3)).astype(np.float32)
    q = r.normal(size=(200, 3)).astype(np.float32)
    idx, d2 = orc.knn(q, v, 19)
    _, ref = cKDTree(v.astype(np.float64)).query(q.astype(np.float64), k=19)
    assert (np.sort(idx, 1) == np.sort(ref, 1)).mean() > 0.999          # library routine (fp64) agrees
    assert np.all(np.diff(d2, axis=1) >= 0)
    # ties: integer lattice, many equal distances -> lower index first (PAPER.md silent; L0)
    g = np.stack(np.meshgrid(*[np.arange(4)] * 3, indexing="ij"), -1).reshape(-1, 3).astype(np.float32)
    idx, d2 = orc.knn(g, g, 7)
    D = ((g[:, None] - g[None]) ** 2).sum(-1)
    ref = np.argsort(D, axis=1, kind="stable")[:, :7]
    assert np.array_equal(idx, ref)
    assert np.array_equal(idx[:, 0], np.arange(len(g)))                 # self is its own nearest (A15)


def test_eq1_weights_hand_example_and_constant_field():
    # u_j = 1/||x_g - x_j||.  Distances 1,2,4 -> u = 1, 1/2, 1/4 -> ubar = 4/7, 2/7, 1/7.
    v = np.array([[1, 0, 0], [0, 2, 0], [0, 0, 4], [9, 9, 9]], np.float32)
    q = np.zeros((1, 3), np.float32)
    idx, d2 = orc.knn(q, v, 3)
    ub = orc.interp_weights(d2)
    assert idx.tolist() == [[0, 1, 2]]
    np.testing.assert_allclose(ub[0], [4 / 7, 2 / 7, 1 / 7], rtol=1e-6)
    attr = np.array([[7.0], [14.0], [28.0], [0.0]], np.float32)
    np.testing.assert_allclose(orc.interp_attr(idx, ub, attr)[0, 0], 4 + 4 + 4, rtol=1e-6)
    r = np.random.default_rng(2)
    v = r.normal(size=(300, 3)).astype(np.float32); q = r.normal(size=(50, 3)).astype(np.float32)
    idx, d2 = orc.knn(q, v, 3); ub = orc.interp_weights(d2)
    np.testing.assert_allclose(ub.sum(1), 1.0, atol=2e-7)
    const = np.full((300, 5), 3.25, np.float32)
    np.testing.assert_allclose(orc.interp_attr(idx, ub, const), 3.25, rtol=3e-7)
    # a Gaussian sitting exactly on a vertex takes that vertex's value (distance clamp, A1)
    idx, d2 = orc.knn(v[:4], v, 3); ub = orc.interp_weights(d2)
    lin = v @ np.array([1.0, 2.0, 3.0], np.float32)
    np.testing.assert_allclose(orc.interp_attr(idx, ub, lin[:, None])[:, 0], lin[:4], rtol=1e-5)


# ------------------------------------------------------------------ H1/H2: skinning
def _rigid(r):
    A = r.normal(size=(3, 3)); Q, _ = np.linalg.qr(A)
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    return np.concatenate([Q, r.normal(size=(3, 1))], 1)


def test_skin_identity_rigid_and_blend():
    r = np.random.default_rng(3)
    n, B = 64, 5
    x = r.normal(size=(n, 3)).astype(np.float32); dx = (0.01 * r.normal(size=(n, 3))).astype(np.float32)
    nr = r.normal(size=(n, 3)); nr = (nr / np.linalg.norm(nr, axis=1, keepdims=True)).astype(np.float32)
    w = r.uniform(size=(n, B)).astype(np.float32); w /= w.sum(1, keepdims=True)
    I = np.tile(np.eye(3, 4).reshape(12), (B, 1)).astype(np.float32)
    xo, no, _ = orc.skin(x, dx, nr, np.eye(B, dtype=np.float32)[r.integers(0, B, n)], I)
    assert np.array_equal(xo, x + dx)                                   # identity pose: bit-exact x + dx
    G = _rigid(r)
    xo, no, M = orc.skin(x, dx, nr, w, np.tile(G.reshape(12), (B, 1)).astype(np.float32))
    xb = (x + dx).astype(np.float64)
    np.testing.assert_allclose(xo, xb @ G[:, :3].T + G[:, 3], atol=2e-6)   # partition of unity
    np.testing.assert_allclose(no, nr.astype(np.float64) @ G[:, :3].T, atol=2e-6)
    # covariance under a rigid bone: eigenvalues = s^2 (rotation invariance, A3)
    q = r.normal(size=(n, 4)).astype(np.float32); s = np.exp(r.uniform(-5, -3, (n, 3))).astype(np.float32)
    c6 = orc.gauss_cov(M, q, s).astype(np.float64)
    S = np.zeros((n, 3, 3)); iu = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
    for k, (a, b) in enumerate(iu):
        S[:, a, b] = c6[:, k]; S[:, b, a] = c6[:, k]
    ev = np.linalg.eigvalsh(S)
    np.testing.assert_allclose(ev, np.sort(s.astype(np.float64) ** 2, 1), rtol=2e-4)
    # two translating bones, weights 1/4, 3/4 -> x + t1/4 + 3 t2/4 (hand example of linear blend)
    G2 = np.tile(np.eye(3, 4), (2, 1, 1)); G2[0, :, 3] = [4, 0, 0]; G2[1, :, 3] = [0, 8, 0]
    xo, _, _ = orc.skin(np.zeros((1, 3), np.float32), None, np.array([[0, 0, 1]], np.float32),
                        np.array([[0.25, 0.75]], np.float32), G2.reshape(2, 12).astype(np.float32))
    assert xo.tolist() == [[1.0, 6.0, 0.0]]


def test_cov_axis_aligned_quaternion():
    # q = (cos 45deg, 0, 0, sin 45deg): rotation by 90deg about z sends x->y: Sigma = diag(s_y^2, s_x^2, s_z^2)
    M = np.eye(3, 4, dtype=np.float32).reshape(1, 12)
    q = np.array([[np.sqrt(0.5), 0, 0, np.sqrt(0.5)]], np.float32)
    c6 = orc.gauss_cov(M, q, np.array([[1.0, 2.0, 3.0]], np.float32))[0]
    np.testing.assert_allclose(c6, [4, 0, 0, 1, 0, 9], atol=1e-5)


# ------------------------------------------------------------------ env quadrature + BRDF + shading
def test_env_quadrature_closed_forms():
    for (R, C) in [(8, 16), (16, 32), (32, 64)]:
        w, A = orc.env_table(R, C)
        np.testing.assert_allclose(A.sum(), 4 * np.pi, rtol=1e-12)      # exact solid angles (A6)
        np.testing.assert_allclose((A[:, None] * w).sum(0), 0, atol=1e-12)
        np.testing.assert_allclose(np.linalg.norm(w, axis=1), 1, atol=1e-12)
    w, A = orc.env_table(16, 32)
    assert w[0, 2] > 0.99 and w[-1, 2] < -0.99                          # row 0 = +z pole (z-up)
    # texel (8,0): theta just past the equator, phi = pi/32
    np.testing.assert_allclose(w[8 * 32], [np.sin(8.5 * np.pi / 16) * np.cos(np.pi / 32),
                                            np.sin(8.5 * np.pi / 16) * np.sin(np.pi / 32), np.cos(8.5 * np.pi / 16)], atol=1e-12)


def test_brdf_normal_incidence_golden():
    # Closed form of Eq.12-15 at w_i = w_o = n: D = 1/(pi a^2), G1 = 1, F = .04 + .96 2^-12.53789
    n = np.array([0, 0, 1.0])
    for rough, spec_gold in _golden("brdf_normal_incidence.txt"):
        R = orc.brdf(n, n, n, np.zeros(3), rough, 1.0)
        np.testing.assert_allclose(R, spec_gold, rtol=2e-4)
    R = orc.brdf(n, n, n, np.array([0.2, 0.4, 0.6]), 0.5, 0.0)
    np.testing.assert_allclose(R, np.array([0.2, 0.4, 0.6]) / np.pi, rtol=1e-12)    # Lambert term a/pi


def test_brdf_reciprocity_ndf_normalisation_fresnel():
    r = np.random.default_rng(5)
    n = np.array([0, 0, 1.0])
    for _ in range(50):
        a = r.normal(size=3); a[2] = abs(a[2]) + 0.05; a /= np.linalg.norm(a)
        b = r.normal(size=3); b[2] = abs(b[2]) + 0.05; b /= np.linalg.norm(b)
        rough = r.uniform(0.1, 1)
        np.testing.assert_allclose(orc.brdf(a, b, n, np.ones(3), rough, 0.7), orc.brdf(b, a, n, np.ones(3), rough, 0.7), rtol=1e-10)
    # NDF normalisation: with w_i = w_o = h,  D(h) = R 4 ((n.h)(1-k)+k)^2 / F(1);  integral D (n.h) dh = 1 (GGX)
    for rough in (0.3, 0.5, 1.0):
        k = (rough + 1) ** 2 / 8
        F1 = 0.04 + 0.96 * 2 ** (-5.55473 - 6.98316)
        th = (np.arange(20000) + 0.5) * (np.pi / 2) / 20000
        D = np.array([orc.brdf(h, h, n, np.zeros(3), rough, 1.0)[0] for h in
                      np.stack([np.sin(th), 0 * th, np.cos(th)], 1)]) * 4 * (np.cos(th) * (1 - k) + k) ** 2 / F1
        integral = (D * np.cos(th) * np.sin(th)).sum() * (np.pi / 2 / 20000) * 2 * np.pi
        np.testing.assert_allclose(integral, 1.0, rtol=2e-4)
    # gamma = 1 -> alpha = 1 -> D = 1/pi for every h
    h = np.array([np.sin(0.7), 0, np.cos(0.7)])
    k = 0.5
    np.testing.assert_allclose(orc.brdf(h, h, n, np.zeros(3), 1.0, 1.0)[0] * 4 * (h[2] * (1 - k) + k) ** 2 / F1, 1 / np.pi, rtol=1e-10)
    # spherical-Gaussian Fresnel stays within 0.004 of Schlick's (1-x)^5 (UE4 approximation, Eq.14)
    x = np.linspace(0, 1, 1001)
    assert np.abs((0.04 + 0.96 * 2 ** ((-5.55473 * x - 6.98316) * x)) - (0.04 + 0.96 * (1 - x) ** 5)).max() < 0.004


def test_white_furnace_lambert():
    # north_star pin: constant white env, full visibility, Lambertian (p = 0): L_o = a E(n) / pi,
    # E(n) = sum_k A_k max(0, n.w_k) by an independent loop; E/pi -> 1 within the quadrature error of the grid.
    r = np.random.default_rng(6)
    n = r.normal(size=(300, 3)); n = (n / np.linalg.norm(n, axis=1, keepdims=True)).astype(np.float32)
    x = (0.1 * r.normal(size=(300, 3))).astype(np.float32)
    alb = r.uniform(size=(300, 3)).astype(np.float32)
    for (R, C, lo, hi) in [(16, 32, 0.995, 1.005), (8, 16, 0.98, 1.02), (32, 64, 0.9985, 1.0015)]:
        env = np.ones((R, C, 3), np.float32)
        Lo, cg = orc.shade(x, n, alb, np.full(300, 0.5, np.float32), np.zeros(300, np.float32), np.array([0, -5, 0], np.float32),
                           env, None, 2)
        th = (np.arange(R) + 0.5) * np.pi / R; ph = (np.arange(C) + 0.5) * 2 * np.pi / C
        E = np.zeros(300)
        for i in range(R):
            A = (np.cos(i * np.pi / R) - np.cos((i + 1) * np.pi / R)) * 2 * np.pi / C
            for j in range(C):
                wk = np.array([np.sin(th[i]) * np.cos(ph[j]), np.sin(th[i]) * np.sin(ph[j]), np.cos(th[i])])
                E += A * np.maximum(0, n.astype(np.float64) @ wk)
        np.testing.assert_allclose(Lo, alb.astype(np.float64) * E[:, None] / np.pi, rtol=1e-9)
        assert lo <= (E / np.pi).min() and (E / np.pi).max() <= hi
        np.testing.assert_allclose(cg, np.clip(Lo, 0, 1) ** (1 / 2.2), rtol=1e-12)       # gamma (A9, unpinned value)


def test_shade_single_light_hand_example():
    # One bright texel, everything else black: L_o = L A R cos (Eq.2 with a single term), visibility bit gates it.
    R_, C_ = 8, 16
    w, A = orc.env_table(R_, C_)
    k = 2 * C_ + 3
    env = np.zeros((R_, C_, 3), np.float32); env[2, 3] = [2.0, 3.0, 4.0]
    n = np.array([[0, 0, 1.0]], np.float32); x = np.zeros((1, 3), np.float32)
    cam = np.array([0, -3.0, 4.0], np.float32); wo = cam / np.linalg.norm(cam)
    alb = np.array([[0.5, 0.6, 0.7]], np.float32)
    Rr = orc.brdf(w[k], wo.astype(np.float64), n[0].astype(np.float64), alb[0].astype(np.float64), 0.4, 0.8)
    bits = np.zeros((1, 4), np.uint32); bits[0, k >> 5] = 1 << (k & 31)
    Lo, _ = orc.shade(x, n, alb, np.array([0.4], np.float32), np.array([0.8], np.float32), cam, env, None, 0, bits=bits, K=128)
    np.testing.assert_allclose(Lo[0], np.array([2.0, 3.0, 4.0]) * A[k] * Rr * w[k, 2], rtol=1e-7)
    Lo0, _ = orc.shade(x, n, alb, np.array([0.4], np.float32), np.array([0.8], np.float32), cam, env, None, 0,
                       bits=np.zeros((1, 4), np.uint32), K=128)
    assert np.all(Lo0 == 0)                                             # shadowed -> no light


# ------------------------------------------------------------------ H3/H4: visibility
def _ray_tri_depth(orig, w, v, f):
    """Nearest hit parameter of rays orig - t*w ... brute-force double Moeller-Trumbore; returns max over w.(p-c)."""
    best = np.full(len(orig), -np.inf)
    hit = np.zeros(len(orig), bool)
    for t in f:
        a, b, c = v[t[0]], v[t[1]], v[t[2]]
        e1, e2 = b - a, c - a
        d = -w
        pv = np.cross(d, e2); det = e1 @ pv
        if abs(det) < 1e-14:
            continue
        tv = orig - a
        uu = (tv @ pv) / det
        qv = np.cross(tv, e1)
        vv = (qv @ d) / det
        tt = (qv @ e2) / det
        ok = (uu >= -1e-9) & (vv >= -1e-9) & (uu + vv <= 1 + 1e-9)
        dep = (orig + tt[:, None] * d) @ w
        upd = ok & (dep > best)
        best[upd] = dep[upd]; hit |= ok
    return best, hit


def test_depth_map_equals_bruteforce_rays_tiny_mesh():
    v, f = smesh.icosphere(1)
    v = (v * np.array([1.0, 0.7, 0.5]) + np.array([0.1, -0.2, 0.3])).astype(np.float32)
    dirs = workloads.latlong_dirs(2, 4)[[0, 3, 5, 6]]
    R = 24
    c, r = orc.window(v)
    zmap, ids = orc.vis_raster(v, f, dirs, R, c, r)
    fr = orc.light_frames(dirs).astype(np.float64)
    vd = v.astype(np.float64)
    for k in range(len(dirs)):
        u, vv, w = fr[k, :3], fr[k, 3:6], fr[k, 6:]
        ii, jj = np.meshgrid(np.arange(R), np.arange(R), indexing="xy")
        pu = ((ii.reshape(-1) + 0.5) / R * 2 - 1) * r; pv = ((jj.reshape(-1) + 0.5) / R * 2 - 1) * r
        orig = c.astype(np.float64) + pu[:, None] * u + pv[:, None] * vv
        dep, hit = _ray_tri_depth(orig, w, vd, f)
        z = zmap[k].reshape(-1); zf = z.view(np.float32).astype(np.float64)
        covered = z != 0xFFFFFFFF
        # coverage agrees except for pixel centres within a subpixel snap of a silhouette edge
        assert (covered != hit).mean() < 0.03
        both = covered & hit
        zref = (r - (dep - c.astype(np.float64) @ w)) / (2 * r)
        err = np.abs(zf[both] - zref[both])
        assert np.quantile(err, 0.97) < 2e-3 and np.median(err) < 2e-4     # snap = 1/256 px of a 24 px map
        assert both.sum() > 50
    assert ids.max() < len(f) and ids.min() >= -1


def test_depth_test_convex_body_pin():
    # Convex body (unposed icosphere): a surface point sees w iff n.w > 0.  One-sided checks (A17).
    inp = workloads.make(0)
    inp["bone_mats"][0] = np.tile(np.eye(3, 4).reshape(12), (2, 1))
    av = orc.avatar_load(inp)
    o = orc.render_frame(av, inp, vis_mode=0, stop_after="vis")
    K = len(inp["vis_dirs"])
    bits = ((o["visbits"][:, :, None] >> np.arange(32)[None, None, :]) & 1).reshape(len(o["visbits"]), -1)[:, :K]
    # outward normal of the sphere at the Gaussian
    nx = o["gauss_posed"] / np.linalg.norm(o["gauss_posed"], axis=1, keepdims=True)
    cs = nx @ inp["vis_dirs"].T
    assert np.all(bits[cs > 0.02] == 1)           # no false self-shadow on the lit side
    assert np.all(bits[cs < -0.4] == 0)           # far side is shadowed
    assert 0.4 < bits.mean() < 0.65


def test_paper_visibility_filters_and_convex_pin(cfg0):
    inp = dict(cfg0); inp["bone_mats"] = cfg0["bone_mats"].copy()
    inp["bone_mats"][0] = np.tile(np.eye(3, 4).reshape(12), (2, 1))
    av = orc.avatar_load(inp)
    o = orc.render_frame(av, inp, vis_mode=1, stop_after="vis")
    nv = len(inp["vert_pos"])
    vcount, (raw, m1, m2) = orc.vis_paper(o["idmap"], inp["faces"], nv, av["knn_v"], want_stages=True)
    assert vcount.max() <= 19 and np.array_equal(vcount, o["vcount"])
    knn = av["knn_v"]
    # brute-force re-evaluation of Eq.3-4 with numpy
    med = lambda V: (V[:, knn].sum(-1) * 2 > knn.shape[1]).astype(np.uint8)
    assert np.array_equal(m1, med(raw)) and np.array_equal(m2, med(m1))
    assert np.array_equal(vcount, m2[:, knn].sum(-1).T)
    # raw bits = "triangle appears in the image -> its three vertices"
    k = 3
    tri = np.unique(o["idmap"][k][o["idmap"][k] >= 0])
    ref = np.zeros(nv, np.uint8); ref[inp["faces"][tri].reshape(-1)] = 1
    assert np.array_equal(raw[k], ref)
    # convex pin: filtered value ~1 on the clearly lit side, exactly 0 on the far side
    cs = inp["vert_normal"] @ inp["vis_dirs"].T
    vbar = vcount / 19.0
    assert vbar[cs > 0.5].min() >= 0.94
    assert np.all(raw.T[cs < -0.1] == 0)          # no triangle facing away ever wins a pixel on a convex body
    assert np.all(vbar[cs < -0.45] == 0)          # the 19-neighbourhood of a 642-vertex sphere spans ~0.35 in n.w
    # fixed points: all-ones / all-zeros maps survive median and mean
    ones = np.full((1, 8, 8), 0, np.int32)          # every pixel won by triangle 0 ...
    allv = orc.vis_paper(np.zeros((1, 4, 4), np.int32) - 1, inp["faces"], nv, knn)
    assert np.all(allv == 0)
    vg = orc.vis_gauss(vcount, av["knn_g"], av["ubar_g"], 19)
    assert vg.min() >= 0 and vg.max() <= 1 + 1e-6


# ------------------------------------------------------------------ H6-H10: splatting
def _one_gauss_inputs(s=0.05, z=4.0, o=0.8, W=64, H=64, f=80.0):
    cam = dict(R_wc=np.eye(3, dtype=np.float32).reshape(9), t_wc=np.zeros(3, np.float32), fx=np.float32(f), fy=np.float32(f),
               cx=np.float32(W / 2), cy=np.float32(H / 2), width=W, height=H, z_near=np.float32(0.2))
    x = np.array([[0, 0, z]], np.float32); n = np.array([[0, 0, -1.0]], np.float32)
    cov = np.array([[s * s, 0, 0, s * s, 0, s * s]], np.float32)
    return cam, x, n, cov, np.array([o], np.float32)


def test_single_isotropic_gaussian_matches_analytic():
    # north_star pin: on-axis isotropic splat = c min(0.99, o exp(-|p-mu|^2 / (2 s'^2))), s'^2 = (f s / z)^2 + 0.3
    s, z, o, W, H, f = 0.05, 4.0, 0.8, 64, 64, 80.0
    cam, x, n, cov, op = _one_gauss_inputs(s, z, o, W, H, f)
    P = orc.project(x, n, cov, op, cam)
    assert P["touched"][0] > 0 and P["depth"][0] == np.float32(z)
    np.testing.assert_allclose(P["mu"][0], [W / 2, H / 2])
    keys, vals = orc.emit_sort(P["depth"], P["rect"], P["touched"], 4)
    rng = orc.tile_ranges(keys, 16)
    col = np.array([[0.9, 0.5, 0.25]])
    img, T, nc, fl = orc.composite(vals, rng, P["mu"], P["conic_o"], col, np.zeros(3, np.float32), W, H)
    sp2 = (f * s / z) ** 2 + 0.3
    yy, xx = np.meshgrid(np.arange(H) + 0.5, np.arange(W) + 0.5, indexing="ij")
    a = np.minimum(0.99, o * np.exp(-((xx - W / 2) ** 2 + (yy - H / 2) ** 2) / (2 * sp2)))
    rad = int(np.ceil(3 * np.sqrt(sp2)))
    assert P["radius"][0] == rad
    x0, x1 = int((W / 2 - rad) // 16), int((W / 2 + rad + 15) // 16)
    tile_ok = ((xx // 16) >= x0) & ((xx // 16) < x1) & ((yy // 16) >= x0) & ((yy // 16) < x1)
    a = np.where((a >= 1 / 255) & tile_ok, a, 0.0)
    np.testing.assert_allclose(img, a[:, :, None] * col[0], atol=2e-6)
    np.testing.assert_allclose(T, 1 - a, atol=2e-6)
    # opacity -> 0 and facing away -> background
    P2 = orc.project(x, -n, cov, op, cam)
    assert P2["touched"][0] == 0


def test_two_gaussian_over_operator_hand_example():
    # front-to-back "over": C = c1 a1 + c2 a2 (1 - a1) at the shared centre pixel sample
    cam, x, n, cov, op = _one_gauss_inputs()
    x2 = np.array([[0, 0, 4.0], [0, 0, 3.0]], np.float32)        # second one is nearer -> composited first
    P = orc.project(x2, np.tile(n, (2, 1)), np.tile(cov, (2, 1)), np.array([0.5, 0.25], np.float32), cam)
    keys, vals = orc.emit_sort(P["depth"], P["rect"], P["touched"], 4)
    rng = orc.tile_ranges(keys, 16)
    col = np.array([[1.0, 0, 0], [0, 1.0, 0]])
    img, T, nc, _ = orc.composite(vals, rng, P["mu"], P["conic_o"], col, np.array([0, 0, 1], np.float32), 64, 64)

    def alpha(g, px, py):
        d = P["mu"][g].astype(np.float64) - [px, py]; c = P["conic_o"][g].astype(np.float64)
        return min(0.99, c[3] * np.exp(-0.5 * (c[0] * d[0] ** 2 + c[2] * d[1] ** 2) - c[1] * d[0] * d[1]))
    a_near, a_far = alpha(1, 32.5, 32.5), alpha(0, 32.5, 32.5)
    np.testing.assert_allclose(img[32, 32], [a_far * (1 - a_near), a_near, (1 - a_near) * (1 - a_far)], rtol=1e-9)
    assert vals[np.searchsorted(keys >> 32, 2 * 4 + 2)] == 1     # nearer Gaussian first in tile (2,2)


def test_tiled_equals_bruteforce_and_invariants(cfg0, cfg0_oracle):
    av, o, o1 = cfg0_oracle
    cam = cfg0["camera"]; W, H = cam["width"], cam["height"]
    img, T, nc = orc.composite_bruteforce(o["depth"], o["rect"], o["touched"], o["mu"], o["conic_o"], o["color"], cfg0["bg"], W, H)
    assert np.array_equal(img, o["image"]) and np.array_equal(T, o["T_final"]) and np.array_equal(nc, o["n_contrib"])
    assert o["T_final"].min() >= 0 and o["T_final"].max() <= 1
    assert o["image"].max() <= o["color"][o["touched"] > 0].max() + 1e-12
    keys, vals = o["keys"], o["vals"]
    assert np.all(np.diff(keys.astype(np.uint64)) >= 0) or np.all(keys[1:] >= keys[:-1])
    assert len(keys) == o["touched"].sum()
    assert np.array_equal(np.bincount(vals, minlength=len(o["touched"])), o["touched"])    # permutation of the emitted list
    same = keys[1:] == keys[:-1]
    assert np.all(vals[1:][same] > vals[:-1][same])                                       # stability (A22)
    r = o["ranges"].astype(np.int64); L = r[:, 1] - r[:, 0]
    assert L.sum() == len(keys)
    nz = r[L > 0]
    assert np.array_equal(nz[1:, 0], nz[:-1, 1]) and nz[0, 0] == 0                        # ranges partition [0, D)
    # black environment -> image = background
    Lo, cg = orc.shade(o["gauss_posed"], o["gauss_normal_posed"], av["albedo_g"], av["rough_g"], av["spec_g"], cfg0["cam_pos"],
                       np.zeros_like(cfg0["env"][0]), cfg0["texel_to_dir"], 2)
    bg = np.array([0.25, 0.5, 0.75], np.float32)
    img0, _, _, _ = orc.composite(o["vals"], o["ranges"], o["mu"], o["conic_o"], cg, bg, W, H)
    np.testing.assert_allclose(img0, np.broadcast_to(bg, img0.shape) * o["T_final"][:, :, None], atol=1e-12)


def test_projection_matches_double_precision_ewa(cfg0, cfg0_oracle):
    # Independent numpy fp64 EWA (J W Sigma W^T J^T + 0.3 I) against the op-ordered fp32 oracle.
    av, o, _ = cfg0_oracle
    cam = cfg0["camera"]
    Rw = cam["R_wc"].reshape(3, 3).astype(np.float64); tw = cam["t_wc"].astype(np.float64)
    g = np.nonzero(o["touched"])[0][:200]
    x = o["gauss_posed"][g].astype(np.float64)
    t = x @ Rw.T + tw
    c6 = o["cov6"][g].astype(np.float64)
    fx, fy = float(cam["fx"]), float(cam["fy"])
    for i in range(len(g)):
        S = np.array([[c6[i, 0], c6[i, 1], c6[i, 2]], [c6[i, 1], c6[i, 3], c6[i, 4]], [c6[i, 2], c6[i, 4], c6[i, 5]]])
        J = np.array([[fx / t[i, 2], 0, -fx * t[i, 0] / t[i, 2] ** 2], [0, fy / t[i, 2], -fy * t[i, 1] / t[i, 2] ** 2]])
        c2 = J @ Rw @ S @ Rw.T @ J.T + 0.3 * np.eye(2)
        con = np.linalg.inv(c2)
        np.testing.assert_allclose(o["conic_o"][g[i], :3], [con[0, 0], con[0, 1], con[1, 1]], rtol=2e-3, atol=1e-5)
        lam = np.linalg.eigvalsh(c2).max()
        assert abs(o["radius"][g[i]] - np.ceil(3 * np.sqrt(lam))) <= 1
        np.testing.assert_allclose(o["mu"][g[i]], [fx * t[i, 0] / t[i, 2] + float(cam["cx"]), fy * t[i, 1] / t[i, 2] + float(cam["cy"])], rtol=1e-5)
    # back-facing Gaussians are culled, front-facing in-frustum ones are kept
    wo = cfg0["cam_pos"].astype(np.float64) - o["gauss_posed"]
    facing = (o["gauss_normal_posed"] * wo).sum(1)
    assert np.all(o["touched"][facing < -1e-4] == 0)
    assert (o["touched"][facing > 1e-4] > 0).mean() > 0.99


# --------------------------------------------------------------------------------------------- displacement network
def _tiny_mlp(width=2, F=1, P=1):
    z = lambda *s: np.zeros(s)
    return dict(rff=np.array([[0.25, 0.0, 0.0]]), W1=z(width, 2 * F + P), b1=z(width), Wh=z(3, width, width), bh=z(3, width),
                Wo=z(3, width), bo=z(3))


def test_disp_mlp_hand_example():
    # PAPER.md:86, :191-193 (readings A26-A28).  x = (1,0,0), B = (0.25,0,0): 2 pi B.x = pi/2, so gamma = (sin, cos) = (1, 0).
    from oracle import oracle as orc
    m = _tiny_mlp()
    m["W1"][:] = [[2.0, 5.0, 3.0], [-1.0, 7.0, 0.0]]           # columns: sin, cos, theta
    m["b1"][:] = [0.5, 0.25]                                   # h1 = relu(2*1 + 3*0.5 + 0.5, -1 + 0.25) = (4, 0)
    for l in range(3):
        m["Wh"][l] = np.eye(2)                                 # identity layers keep (4, 0)
    m["bh"][2] = [1.0, -1.0]                                   # last hidden: relu(5, -1) = (5, 0)
    m["Wo"][:] = [[1.0, 9.0], [0.5, 9.0], [-2.0, 9.0]]; m["bo"][:] = [0.0, 1.0, 2.0]
    dx = orc.disp_mlp(np.array([[1.0, 0.0, 0.0]]), np.array([0.5]), m)
    assert np.allclose(dx, [[5.0, 3.5, -8.0]], atol=1e-12)


def test_disp_mlp_relu_and_affine_regime():
    from oracle import oracle as orc
    from synth import workloads
    m = workloads.make_disp_mlp(seed=3)
    m64 = {k: (np.asarray(v, np.float64) if isinstance(v, np.ndarray) else v) for k, v in m.items()}
    x = np.random.default_rng(0).uniform(-1, 1, (50, 3))
    # all first-layer pre-activations negative: every hidden unit is dead, dx = W_o relu(b_4 ...) is the same for all x
    dead = dict(m64); dead["b1"] = m64["b1"] - 1e3
    dx = orc.disp_mlp(x, m64["theta"], dead)
    h = np.maximum(m64["bh"][0], 0.0)
    for l in (1, 2):
        h = np.maximum(m64["Wh"][l] @ h + m64["bh"][l], 0.0)
    assert np.allclose(dx, np.broadcast_to(m64["Wo"] @ h + m64["bo"], dx.shape), atol=1e-12)
    # all pre-activations positive (a large first bias, non-negative hidden weights and biases): no ReLU clips, the
    # network is affine, dx = W_o W_4 W_3 W_2 (W_1 h0 + b1) + ... composed by hand
    aff = dict(m64); aff["b1"] = m64["b1"] + 1e3; aff["Wh"] = np.abs(m64["Wh"]); aff["bh"] = np.abs(m64["bh"]) + 1.0
    p = 2 * np.pi * x @ m64["rff"].T
    h0 = np.concatenate([np.sin(p), np.cos(p), np.broadcast_to(m64["theta"], (50, 72))], 1)
    A, c = aff["W1"], aff["b1"]
    for l in range(3):
        A, c = aff["Wh"][l] @ A, aff["Wh"][l] @ c + aff["bh"][l]
    A, c = aff["Wo"] @ A, aff["Wo"] @ c + aff["bo"]
    assert np.allclose(orc.disp_mlp(x, m64["theta"], aff), h0 @ A.T + c, rtol=1e-9, atol=1e-6)
    # gamma(x) is 1-periodic along B's rows: shifting x by a vector v with B v integer leaves dx unchanged
    Bm = np.zeros_like(m64["rff"]); Bm[:, 0] = np.arange(1, 65)            # integer frequencies along x
    per = dict(m64); per["rff"] = Bm
    assert np.allclose(orc.disp_mlp(x, m64["theta"], per), orc.disp_mlp(x + np.array([1.0, 0.3, -2.0]), m64["theta"], per), atol=1e-9)


# ------------------------------------------------------------------ Algorithm 1: density-based densification
def _tiny_densify_case():
    # a strip of 4 triangles over 6 vertices; 5 Gaussians with hand-written K_g = 3 neighbour sets
    x = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [1, 1, 0], [0, 2, 0], [1, 2, 0]], np.float32)
    faces = np.array([[0, 1, 2], [1, 3, 2], [2, 3, 4], [3, 5, 4]], np.int32)
    knn = np.array([[0, 1, 2], [0, 1, 2], [1, 2, 3], [0, 2, 1], [2, 1, 0]], np.int32)
    return x, faces, knn


def test_densify_hand_example_counts_density_and_budget():
    # PAPER.md:489-503 by hand.  D_v = occurrences of each vertex in S_g: v0 4, v1 5, v2 5, v3 1, v4 0, v5 0.
    # d_f = (sum of the three D_v) / (6 K_g = 18): 14/18, 11/18, 6/18, 1/18.  With d_0 = 1: P = 4/18, 7/18, 12/18, 17/18,
    # sum(P) = 40/18; N' = floor(sum(P) p_0) = floor(2.222 * 0.9) = 2 (the algorithm's "sum(P) x p_0").
    x, faces, knn = _tiny_densify_case()
    rnd = np.zeros(3 * 8, np.uint32)
    r = orc.densify_density(knn, faces, x, 1.0, 0.9, rnd)
    assert r["D_v"].tolist() == [4, 5, 5, 1, 0, 0]
    assert r["D_v"].sum() == knn.size                                      # every (Gaussian, neighbour) pair counted once
    assert np.allclose(r["P_fix"] / 65536.0, np.array([4, 7, 12, 17]) / 18.0, atol=2.0 ** -17)
    assert r["n_add"] == 2 and len(r["tri"]) == 2 and r["n_g"].sum() == 2
    # a triangle at or above the threshold gets probability 0 ("below d_0")
    r = orc.densify_density(knn, faces, x, 0.5, 0.9, rnd)
    assert r["P_fix"][0] == 0 and r["P_fix"][1] == 0 and r["P_fix"][2] > 0
    # "we need a total of sum(P) Gaussians ... but only add a small percent p_0" (:477): p_0 = 1 asks for floor(sum(P))
    assert orc.densify_density(knn, faces, x, 1.0, 1.0, rnd)["n_add"] == 2
    assert orc.densify_density(knn, faces, x, 4.0, 1.0, rnd)["n_add"] == int(np.floor(4 * 4 - 32 / 18.0))


def test_densify_multinomial_extremes_and_frequencies():
    x, faces, knn = _tiny_densify_case()
    n = 40000
    # inverse CDF end points: u = 0 picks the first triangle with P > 0, u -> 1 the last
    lo = np.zeros(3 * 4, np.uint32); hi = np.full(3 * 4, 2 ** 32 - 1, np.uint32)
    assert set(orc.densify_density(knn, faces, x, 1.0, 1.9, lo)["tri"].tolist()) == {0}
    assert set(orc.densify_density(knn, faces, x, 1.0, 1.9, hi)["tri"].tolist()) == {3}
    assert set(orc.densify_density(knn, faces, x, 0.5, 5.0, lo)["tri"].tolist()) == {2}     # triangles 0, 1 have P = 0
    # frequencies follow P / sum(P) (multinomial): chi-square against the hand-computed P
    rnd = np.random.default_rng(3).integers(0, 2 ** 32, size=3 * n, dtype=np.uint64).astype(np.uint32)
    r = orc.densify_density(knn, faces, x, 1.0, 1e9, rnd)           # budget far above n: all n draws are made
    assert len(r["tri"]) == n and r["n_g"].sum() == n
    assert np.array_equal(r["n_g"], np.bincount(r["tri"], minlength=4))
    expect = n * np.array([4, 7, 12, 17]) / 40.0
    chi2 = (((r["n_g"] - expect) ** 2) / expect).sum()
    assert chi2 < 25.0                                                # 3 dof: P(chi2 > 25) ~ 1.5e-5


def test_densify_placement_is_uniform_on_the_triangle():
    # one triangle, no Gaussians anywhere: all draws land on it; the points are uniform over its area (:479 "randomly
    # place").  Uniform-on-triangle moments: E[b_i] = 1/3, E[b_i^2] = 1/6, E[b_i b_j] = 1/12.
    x = np.array([[0.2, 0.1, 0.3], [1.3, 0.4, -0.2], [0.1, 1.7, 0.9]], np.float32)
    faces = np.array([[0, 1, 2]], np.int32)
    knn = np.zeros((0, 3), np.int32)
    n = 60000
    rnd = np.random.default_rng(4).integers(0, 2 ** 32, size=3 * n, dtype=np.uint64).astype(np.uint32)
    r = orc.densify_density(knn, faces, x, 1.0, 1e9, rnd)
    assert len(r["pos"]) == n and np.all(r["tri"] == 0)
    A = np.concatenate([x.astype(np.float64).T, np.ones((1, 3))], 0)          # solve for barycentric coordinates
    b = np.linalg.lstsq(A, np.concatenate([r["pos"].astype(np.float64).T, np.ones((1, n))], 0), rcond=None)[0].T
    assert b.min() > -1e-6 and np.allclose(b.sum(1), 1.0, atol=1e-6)          # inside the triangle, on its plane
    assert np.allclose(b.mean(0), 1 / 3, atol=4e-3)
    assert np.allclose((b ** 2).mean(0), 1 / 6, atol=4e-3)
    assert np.allclose([(b[:, 0] * b[:, 1]).mean(), (b[:, 0] * b[:, 2]).mean(), (b[:, 1] * b[:, 2]).mean()], 1 / 12, atol=4e-3)
    # corners of the random square map to corners / edges of the triangle
    c = orc.densify_density(knn, faces, x, 1.0, 1e9, np.array([0, 0, 0, 0, 2 ** 32 - 1, 0], np.uint32))["pos"]
    assert np.allclose(c[0], x[0]) and np.allclose(c[1], x[1], atol=1e-3)


def test_densify_uniform_density_closed_form():
    # regular situation the algorithm's "each vertex is connected with 6 triangles" assumes (:497): every vertex has the
    # same count D -> d_f = 3 D / (6 K_g) = D / (2 K_g) on every triangle, N' = floor(N_f (d_0 - D / (2 K_g)) p_0)
    ico = smesh.icosphere(2)
    x, faces = ico[0], ico[1]
    nv = len(x)
    D, Kg = 2, 3
    knn = np.stack([np.repeat(np.arange(nv), D)] * 3, 1).astype(np.int32)  # N_g = D N_v rows (k, k, k): D_v = 3 D
    r = orc.densify_density(knn, faces, x, 2.0, 0.25, np.zeros(3, np.uint32))
    assert np.all(r["D_v"] == 3 * D)
    d_f = 3 * (3 * D) / (6.0 * Kg)
    assert np.allclose(r["P_fix"] / 65536.0, 2.0 - d_f, atol=2.0 ** -16)
    assert r["n_add"] == int(np.floor(len(faces) * (2.0 - d_f) * 0.25))


def test_backface_cull_option_of_the_depth_rasteriser(cfg0):
    # reading A36: cull = the same rasteriser over the mesh WITHOUT the triangles whose snapped light-space area is
    # negative.  The area is recomputed here in numpy from the light frame (independent of the C++ code path).
    inp = cfg0
    av = orc.avatar_load(inp)
    o = orc.render_frame(av, inp, stop_after="skin")
    dirs, R = inp["vis_dirs"][:24], 64
    xp, f = o["vert_posed"], inp["faces"]
    zc, ic = orc.vis_raster(xp, f, dirs, R, o["win_c"], o["win_r"], cull=True)
    zn, idn = orc.vis_raster(xp, f, dirs, R, o["win_c"], o["win_r"], cull=False)
    uvw = orc.light_frames(dirs)                                        # [K, 9]: u, v, w of every direction
    n_front = 0
    for k in range(len(dirs)):
        s = (R / 2.0) / float(o["win_r"])
        d = (xp - o["win_c"]).astype(np.float64)
        X = np.rint((d @ uvw[k, 0:3].astype(np.float64) * s + R / 2) * 256); Y = np.rint((d @ uvw[k, 3:6].astype(np.float64) * s + R / 2) * 256)
        area = (X[f[:, 1]] - X[f[:, 0]]) * (Y[f[:, 2]] - Y[f[:, 0]]) - (Y[f[:, 1]] - Y[f[:, 0]]) * (X[f[:, 2]] - X[f[:, 0]])
        keep = np.nonzero(area > 0)[0]
        n_front += len(keep)
        zk, ik = orc.vis_raster(xp, f[keep], dirs[k:k + 1], R, o["win_c"], o["win_r"], cull=False)
        assert np.array_equal(zk[0], zc[k])
        assert np.array_equal(np.where(ik[0] >= 0, keep[np.maximum(ik[0], 0)], -1), ic[k])
        # outward-oriented closed mesh: a positive snapped area is a triangle that faces the light
        nrm = np.cross(xp[f[:, 1]] - xp[f[:, 0]], xp[f[:, 2]] - xp[f[:, 0]])
        front = (nrm @ dirs[k]) > 0
        big = np.abs(area) > 4 * 256
        assert (front[big] == (area[big] > 0)).all()
    assert 0.3 < n_front / (len(dirs) * len(f)) < 0.7
    # on a closed mesh the nearest surface is a front face: the culled map differs from the full one only where a nearly
    # edge-on back face extrapolates its plane in front of it (a fraction of a percent of the covered texels)
    cov = zn != 0xFFFFFFFF
    assert np.array_equal(cov, zc != 0xFFFFFFFF)
    assert (zc != zn).sum() < 0.01 * cov.sum()
    assert (zc.view(np.float32)[cov] >= zn.view(np.float32)[cov]).all()
