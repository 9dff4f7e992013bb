"""Pins for the backward oracle (oracle/backward.py): its forward against the independent C++ forward oracle, its
gradients against finite differences taken THROUGH the C++ oracle, hand-derived closed forms, and gradcheck.  No GPU."""
import numpy as np
import pytest
import torch

from oracle import backward as bwd
from oracle import oracle as orc
from synth import workloads


@pytest.fixture(scope="module")
def scene0():
    inp = workloads.make(0)
    av = orc.avatar_load(inp)
    o = orc.render_frame(av, inp, vis_mode=0)
    cam = inp["camera"]
    G = workloads.make_image_cotangent(3, cam["width"], cam["height"])
    r = bwd.splat_backward(o["gauss_posed"], o["cov6"], o["color"], inp["gauss_opacity"], cam, inp["bg"], o["vals"], o["ranges"],
                           o["touched"], G, mu32=o["mu"], conic32=o["conic_o"])
    return inp, o, G, r


def test_backward_oracle_forward_equals_cpp_oracle(scene0):
    inp, o, G, r = scene0
    # stage 1 blends the C++ oracle's own fp32 mu / conic: same decisions, same image (both fp64 blends)
    assert np.array_equal(r["n_contrib"], o["n_contrib"])
    assert np.abs(r["image"] - o["image"]).max() < 1e-12
    assert np.abs(r["T_final"] - o["T_final"]).max() < 1e-12
    # the fp64 projection written in torch agrees with orc_project (fp32 arithmetic) on every surviving Gaussian
    alive = o["touched"] > 0
    mu, conic = bwd.project_torch(torch.as_tensor(o["gauss_posed"][alive].astype(np.float64)),
                                  torch.as_tensor(o["cov6"][alive].astype(np.float64)), inp["camera"])
    assert np.abs(mu.numpy() - o["mu"][alive]).max() < 2e-3                       # pixels, fp32 rounding of ~1e2 px values
    assert np.allclose(conic.numpy(), o["conic_o"][alive, :3], rtol=2e-3, atol=1e-5)
    # without the override the decisions come from the fp64 projection: still the same image to fp32 rounding of mu
    cam = inp["camera"]
    r2 = bwd.splat_backward(o["gauss_posed"], o["cov6"], o["color"], inp["gauss_opacity"], cam, inp["bg"], o["vals"], o["ranges"],
                            o["touched"], G)
    assert np.abs(r2["image"] - o["image"]).max() < 1e-4
    assert np.abs(r2["d_col"] - r["d_col"]).max() < 1e-3 * np.abs(r["d_col"]).max()


def _loss_cpp(o, inp, G, mu=None, conic_o=None, col=None):
    cam = inp["camera"]
    img, _, _, _ = orc.composite(o["vals"], o["ranges"], o["mu"] if mu is None else mu, o["conic_o"] if conic_o is None else conic_o,
                                 o["color"] if col is None else col, inp["bg"], cam["width"], cam["height"])
    return float((img * G).sum())


def test_stage1_gradients_match_finite_differences_through_cpp_composite(scene0):
    # perturbations are exactly representable in fp32 (the C++ blend takes fp32 mu / conic and works in fp64)
    inp, o, G, r = scene0
    rs = np.random.default_rng(0)
    score = np.abs(r["d_mu"]).sum(1) + np.abs(r["d_conic"]).sum(1)
    pick = np.argsort(-score)[:40][rs.permutation(40)[:10]]
    ok = 0
    for g in pick:
        for name, arr, grad, comps in (("mu", o["mu"], r["d_mu"], 2), ("conic", o["conic_o"], r["d_conic"], 3), ("opac", o["conic_o"], r["d_opac"], 1)):
            for c in range(comps):
                col = 3 if name == "opac" else c
                a_p, a_m = arr.copy(), arr.copy()
                h = np.float32(2.0 ** -9) if name == "mu" else np.float32(abs(arr[g, col]) * 2.0 ** -9 + 1e-6)
                a_p[g, col] = arr[g, col] + h; a_m[g, col] = arr[g, col] - h
                kw = "mu" if name == "mu" else "conic_o"
                fd = (_loss_cpp(o, inp, G, **{kw: a_p}) - _loss_cpp(o, inp, G, **{kw: a_m})) / (float(a_p[g, col]) - float(a_m[g, col]))
                an = grad[g] if name == "opac" else grad[g, c]
                if name == "opac" and arr[g, 3] + h > 0.99:
                    continue                                              # opacity 1: alpha clamps for part of the footprint, FD is one-sided
                if abs(fd - an) <= 2e-2 * abs(an) + 2e-3 * np.abs(grad).max():
                    ok += 1
                else:                                                     # a frozen decision flipped under the perturbation: rare
                    ok -= 5
    assert ok > 30
    # colour is linear: finite differences are exact
    for g in pick[:4]:
        for c in range(3):
            cp = o["color"].astype(np.float64).copy(); cp[g, c] += 0.25
            fd = (_loss_cpp(o, inp, G, col=cp) - _loss_cpp(o, inp, G)) / 0.25
            assert abs(fd - r["d_col"][g, c]) < 1e-9 * (1 + abs(fd))


def test_stage2_gradients_match_finite_differences_through_cpp_projection(scene0):
    # L2 = <d_mu, mu(x, Sigma)> + <d_conic, conic(x, Sigma)> through orc_project (fp32 arithmetic -> coarse steps, 1 % tolerance)
    inp, o, G, r = scene0
    cam = inp["camera"]

    def L2(x, cov):
        p = orc.project(x, o["gauss_normal_posed"], cov, inp["gauss_opacity"], cam)
        return (p["mu"].astype(np.float64) * r["d_mu"]).sum(1) + (p["conic_o"][:, :3].astype(np.float64) * r["d_conic"]).sum(1)   # per Gaussian

    alive = np.nonzero(o["touched"] > 0)[0]
    x0, c0 = o["gauss_posed"].astype(np.float32), o["cov6"].astype(np.float32)
    for c in range(3):
        xp, xm = x0.copy(), x0.copy(); xp[:, c] += np.float32(1e-3); xm[:, c] -= np.float32(1e-3)
        fd = (L2(xp, c0) - L2(xm, c0)) / (xp[:, c].astype(np.float64) - xm[:, c])
        err = np.abs(fd[alive] - r["d_x"][alive, c])
        assert np.median(err / (np.abs(r["d_x"][alive, c]) + 1e-3 * np.abs(r["d_x"]).max())) < 1e-2
        assert (err < 3e-2 * np.abs(r["d_x"][alive, c]) + 3e-3 * np.abs(r["d_x"]).max()).mean() > 0.97
    for c in range(6):
        h = (np.abs(c0).max(1) * 0.02).astype(np.float32)
        cp, cm = c0.copy(), c0.copy(); cp[:, c] += h; cm[:, c] -= h
        fd = (L2(x0, cp) - L2(x0, cm)) / (cp[:, c].astype(np.float64) - cm[:, c])
        err = np.abs(fd[alive] - r["d_cov6"][alive, c])
        assert (err < 3e-2 * np.abs(r["d_cov6"][alive, c]) + 3e-3 * np.abs(r["d_cov6"]).max()).mean() > 0.97


def test_one_and_two_gaussian_closed_forms():
    # I = c a + (1 - a) bg,  a = o exp(p),  p = -1/2 (A dx^2 + C dy^2) - B dx dy,  d = mu - pixel   (hand derivatives)
    t = lambda v: torch.tensor(v, dtype=torch.float64, requires_grad=True)
    mu, conic, o, col = t([[5.2, 7.9]]), t([[0.31, 0.07, 0.22]]), t([0.8]), t([[0.9, 0.2, 0.4]])
    bg = torch.tensor([0.1, 0.3, 0.2], dtype=torch.float64); G = np.array([0.7, -1.1, 0.4])
    C, T, n = bwd.composite_tile(mu, conic, o, col, torch.tensor([0]), torch.tensor([4.5], dtype=torch.float64),
                                 torch.tensor([6.5], dtype=torch.float64), bg)
    (C * torch.as_tensor(G)).sum().backward()
    dx, dy = 5.2 - 4.5, 7.9 - 6.5
    p = -0.5 * (0.31 * dx * dx + 0.22 * dy * dy) - 0.07 * dx * dy
    a = 0.8 * np.exp(p)
    s = float(((np.array([0.9, 0.2, 0.4]) - bg.numpy()) * G).sum())
    assert int(n[0]) == 1 and abs(float(T[0].detach()) - (1 - a)) < 1e-15
    assert np.allclose(col.grad.numpy()[0], a * G)
    assert np.isclose(o.grad.item(), np.exp(p) * s)
    assert np.allclose(mu.grad.numpy()[0], [a * s * -(0.31 * dx + 0.07 * dy), a * s * -(0.22 * dy + 0.07 * dx)])
    assert np.allclose(conic.grad.numpy()[0], [a * s * -0.5 * dx * dx, a * s * -dx * dy, a * s * -0.5 * dy * dy])
    # two Gaussians at the same pixel: dI/da1 = c1 - c2 a2 - (1 - a2) bg;  dI/da2 = (1 - a1)(c2 - bg)
    mu, conic = t([[4.5, 6.5], [4.5, 6.5]]), t([[1, 0, 1.0], [1, 0, 1.0]])
    o, col = t([0.6, 0.5]), t([[1.0, 0.0, 0.0], [0.0, 1.0, 0.0]])
    C, T, n = bwd.composite_tile(mu, conic, o, col, torch.tensor([0, 1]), torch.tensor([4.5], dtype=torch.float64),
                                 torch.tensor([6.5], dtype=torch.float64), bg)
    (C * torch.as_tensor(G)).sum().backward()
    c1, c2, b = np.array([1.0, 0, 0]), np.array([0, 1.0, 0]), bg.numpy()
    assert np.allclose(o.grad.numpy(), [((c1 - c2 * 0.5 - 0.5 * b) * G).sum(), (0.4 * (c2 - b) * G).sum()])
    assert np.allclose(col.grad.numpy(), [0.6 * G, 0.4 * 0.5 * G])
    # clamp (reading A32): o exp(p) = 1.2 > 0.99 -> alpha = 0.99 and no gradient reaches o, mu or the conic
    mu, conic, o, col = t([[4.5, 6.5]]), t([[1, 0, 1.0]]), t([1.2]), t([[0.9, 0.2, 0.4]])
    C, T, n = bwd.composite_tile(mu, conic, o, col, torch.tensor([0]), torch.tensor([4.5], dtype=torch.float64),
                                 torch.tensor([6.5], dtype=torch.float64), bg)
    (C * torch.as_tensor(G)).sum().backward()
    assert abs(float(T[0].detach()) - 0.01) < 1e-15 and o.grad.item() == 0.0 and np.all(conic.grad.numpy() == 0) and np.allclose(col.grad.numpy()[0], 0.99 * G)


def test_projection_closed_form_and_gradcheck():
    # identity camera, isotropic Sigma = s2 I: cov2D_xx = (fx / z)^2 s2 (1 + (x/z)^2) + 0.3 on the x axis; mu_x = fx x / z + cx
    cam = {"R_wc": np.eye(3), "t_wc": np.zeros(3), "fx": 100.0, "fy": 100.0, "cx": 32.0, "cy": 32.0, "width": 64, "height": 64, "z_near": 0.1}
    x = torch.tensor([[0.2, 0.0, 2.0]], dtype=torch.float64, requires_grad=True)
    s2 = 0.01
    cov = torch.tensor([[s2, 0, 0, s2, 0, s2]], dtype=torch.float64, requires_grad=True)
    mu, conic = bwd.project_torch(x, cov, cam)
    assert np.allclose(mu.detach().numpy(), [[100 * 0.2 / 2 + 32, 32.0]])
    cxx = (100 / 2.0) ** 2 * s2 * (1 + 0.1 ** 2) + 0.3; cyy = (100 / 2.0) ** 2 * s2 + 0.3
    assert np.allclose(conic.detach().numpy(), [[1 / cxx, 0.0, 1 / cyy]])
    mu[0, 0].backward(retain_graph=True)
    assert np.allclose(x.grad.numpy(), [[100 / 2.0, 0, -100 * 0.2 / 4.0]])          # d mu_x / d(x, y, z)
    x.grad = None; cov.grad = None
    conic[0, 2].backward()
    assert np.allclose(cov.grad.numpy()[0, 3], -(1 / cyy) ** 2 * (100 / 2.0) ** 2)   # d(1/cyy)/d Sigma_yy
    assert np.allclose(cov.grad.numpy()[0, [0, 1, 2]], 0.0)
    # gradcheck of projection + blend on a tiny scene kept away from every threshold
    rs = np.random.default_rng(2)
    n = 5
    X = torch.tensor(np.c_[rs.uniform(-0.05, 0.05, (n, 2)) - [[0.24, 0.24]], rs.uniform(1.8, 2.2, n)], dtype=torch.float64, requires_grad=True)
    A = rs.normal(size=(n, 3, 3)) * 0.02
    S = A @ A.transpose(0, 2, 1) + 0.02 ** 2 * np.eye(3)
    COV = torch.tensor(np.stack([S[:, 0, 0], S[:, 0, 1], S[:, 0, 2], S[:, 1, 1], S[:, 1, 2], S[:, 2, 2]], 1), dtype=torch.float64, requires_grad=True)
    COL = torch.tensor(rs.uniform(0, 1, (n, 3)), dtype=torch.float64, requires_grad=True)
    OP = torch.tensor(rs.uniform(0.3, 0.6, n), dtype=torch.float64, requires_grad=True)
    ys, xs = np.meshgrid(np.arange(16), np.arange(16), indexing="ij")
    px, py = torch.tensor(xs.reshape(-1) + 0.5, dtype=torch.float64), torch.tensor(ys.reshape(-1) + 0.5, dtype=torch.float64)
    sel = torch.tensor([17, 40, 100, 119, 136, 200])
    bg = torch.tensor([0.1, 0.3, 0.2], dtype=torch.float64)

    def f(X, COV, COL, OP):
        mu, conic = bwd.project_torch(X, COV, cam)
        C, T, nc = bwd.composite_tile(mu, conic, OP, COL, torch.arange(n), px[sel], py[sel], bg)
        return C

    assert torch.autograd.gradcheck(f, (X, COV, COL, OP), eps=1e-7, atol=1e-6, rtol=1e-4)


# ------------------------------------------------------------------------------------------------ H5 backward
@pytest.fixture(scope="module")
def shade0():
    inp = workloads.make(0)
    av = orc.avatar_load(inp)
    o = orc.render_frame(av, inp, vis_mode=0)
    env = inp["env"][inp["env_of_frame"][0]]
    N = len(inp["gauss_pos"]); ne = env.shape[0] * env.shape[1]
    v = bwd.texel_visibility(N, ne, inp["texel_to_dir"], 0, bits=o["visbits"])
    d_col = workloads.make_color_cotangent(5, N)
    r = bwd.shade_backward(o["gauss_posed"], o["gauss_normal_posed"], av["albedo_g"], av["rough_g"], av["spec_g"], inp["cam_pos"], env, v,
                           inp["gamma"], d_col)
    return inp, av, o, env, v, d_col, r


def test_shade_backward_oracle_forward_equals_cpp_oracle(shade0):
    inp, av, o, env, v, d_col, r = shade0
    assert np.abs(r["Lo"] - o["L_o"]).max() < 1e-12 and np.abs(r["color"] - o["color"]).max() < 1e-12
    # the paper's visibility (mode 1: fractional v_g) through the same function
    o1 = orc.render_frame(av, inp, vis_mode=1)
    v1 = bwd.texel_visibility(len(v), v.shape[1], inp["texel_to_dir"], 1, vg=o1["vis_g"])
    r1 = bwd.shade_backward(o1["gauss_posed"], o1["gauss_normal_posed"], av["albedo_g"], av["rough_g"], av["spec_g"], inp["cam_pos"], env, v1,
                            inp["gamma"], d_col)
    assert np.abs(r1["Lo"] - o1["L_o"]).max() < 1e-12


def test_shade_gradients_match_finite_differences_through_cpp_shade(shade0):
    inp, av, o, env, v, d_col, r = shade0
    base = dict(xg=o["gauss_posed"].astype(np.float32), ng=o["gauss_normal_posed"].astype(np.float32), alb=av["albedo_g"].astype(np.float32),
                rough=av["rough_g"].astype(np.float32), spec=av["spec_g"].astype(np.float32), env=env.astype(np.float32))

    def loss(**kw):
        a = dict(base); a.update(kw)
        Lo, col = orc.shade(a["xg"], a["ng"], a["alb"], a["rough"], a["spec"], inp["cam_pos"], a["env"], inp["texel_to_dir"], 0,
                            bits=o["visbits"], K=len(inp["vis_dirs"]), gamma=inp["gamma"])
        return (col * d_col).sum(1)                                      # per Gaussian: they are independent

    lit = np.nonzero((o["L_o"] > 1e-3).all(1) & (o["L_o"] < 0.98).all(1))[0]          # away from the clamp limits
    for key, grad, h in (("xg", r["d_x"], 2.0 ** -10), ("ng", r["d_n"], 2.0 ** -12), ("alb", r["d_alb"], 2.0 ** -10),
                         ("rough", r["d_rough"], 2.0 ** -12), ("spec", r["d_spec"], 2.0 ** -10)):
        arr = base[key]
        for c in range(arr.shape[1] if arr.ndim == 2 else 1):
            ap, am = arr.copy(), arr.copy()
            if arr.ndim == 2:
                ap[:, c] += np.float32(h); am[:, c] -= np.float32(h)
                step = ap[:, c].astype(np.float64) - am[:, c]; an = grad[:, c]
            else:
                ap += np.float32(h); am -= np.float32(h)
                step = ap.astype(np.float64) - am; an = grad
            fd = (loss(**{key: ap}) - loss(**{key: am})) / step
            err = np.abs(fd[lit] - an[lit])
            good = err < 2e-3 * np.abs(an[lit]) + 2e-4 * np.abs(an[lit]).max()
            assert good.mean() > 0.98, (key, c, good.mean())              # the few misses: a texel's w_i.n changes sign inside the step
    # environment: L is linear in it up to the gamma curve; perturb single texels
    rs = np.random.default_rng(1)
    for _ in range(6):
        i, j, c = rs.integers(env.shape[0]), rs.integers(env.shape[1]), rs.integers(3)
        ep, em = base["env"].copy(), base["env"].copy(); ep[i, j, c] += np.float32(2.0 ** -8); em[i, j, c] -= np.float32(2.0 ** -8)
        fd = (loss(env=ep)[lit].sum() - loss(env=em)[lit].sum()) / (float(ep[i, j, c]) - float(em[i, j, c]))
        rl = bwd.shade_backward(base["xg"][lit], base["ng"][lit], base["alb"][lit], base["rough"][lit], base["spec"][lit], inp["cam_pos"], env,
                                v[lit], inp["gamma"], d_col[lit])
        assert abs(fd - rl["d_env"][i, j, c]) < 2e-3 * abs(fd) + 1e-4 * np.abs(rl["d_env"]).max()


def test_shade_backward_lambert_closed_form_and_clamp():
    # spec = 0, v = 1, gamma = 1: colour = L_o = a / pi * E(n), E = sum_k L_k A_k max(0, w_k.n)  (the white-furnace pin's
    # setting).  Hand derivatives: d/da = g E / pi, d/dL_k = g a A_k (w_k.n)^+ / pi, d/dn = g a / pi sum_{w_k.n > 0} L_k A_k w_k
    rows, cols = 8, 16
    W, A = orc.env_table(rows, cols)
    rs = np.random.default_rng(3)
    env = rs.uniform(0.05, 0.3, (rows, cols, 3))
    n = np.array([[0.3, -0.5, 0.81]]); n /= np.linalg.norm(n)
    x = np.array([[0.1, 0.2, 0.3]]); alb = np.array([[0.5, 0.6, 0.7]]); g = np.array([[0.7, -0.4, 1.1]])
    r = bwd.shade_backward(x, n, alb, np.array([0.5]), np.array([0.0]), np.array([0.0, -3.0, 0.5]), env, np.ones((1, rows * cols)), 1.0, g)
    cs = np.maximum(W @ n[0], 0.0)
    E = (env.reshape(-1, 3) * (A * cs)[:, None]).sum(0)
    assert np.allclose(r["Lo"][0], alb[0] / np.pi * E)
    assert np.allclose(r["d_alb"][0], g[0] * E / np.pi)
    assert np.allclose(r["d_env"].reshape(-1, 3), (A * cs)[:, None] * (alb[0] * g[0])[None, :] / np.pi)
    assert np.allclose(r["d_n"][0], ((env.reshape(-1, 3) * (alb[0] * g[0])[None, :]).sum(1) * A * (cs > 0)) @ W / np.pi)
    assert np.allclose(r["d_x"][0], 0.0) and r["d_spec"][0] != 0.0      # Lambert term ignores w_o; the specular slot still has slope
    # clamp (reading A33): radiance above 1 (or 0) has colour 1 (0) and no gradient at all
    r = bwd.shade_backward(x, n, alb, np.array([0.5]), np.array([0.0]), np.array([0.0, -3.0, 0.5]), env * 100.0, np.ones((1, rows * cols)), 2.2, g)
    assert np.all(r["color"] == 1.0) and not r["d_alb"].any() and not r["d_env"].any()
    r = bwd.shade_backward(x, n, alb, np.array([0.5]), np.array([0.3]), np.array([0.0, -3.0, 0.5]), env, np.zeros((1, rows * cols)), 2.2, g)
    assert np.all(r["color"] == 0.0) and not r["d_alb"].any() and not r["d_n"].any()


def test_shade_backward_gradcheck():
    rows, cols = 4, 8
    Wn, An = orc.env_table(rows, cols)
    rs = np.random.default_rng(4)
    m = 3
    t = lambda a: torch.tensor(a, dtype=torch.float64, requires_grad=True)
    nn = rs.normal(size=(m, 3)); nn /= np.linalg.norm(nn, axis=1, keepdims=True)
    args = (t(rs.normal(size=(m, 3)) * 0.2), t(nn), t(rs.uniform(0.2, 0.8, (m, 3))), t(rs.uniform(0.3, 0.8, m)), t(rs.uniform(0.2, 0.8, m)))
    env = t(rs.uniform(0.05, 0.2, (rows * cols, 3)))
    cam = torch.tensor([0.3, -2.5, 0.4], dtype=torch.float64)
    v = torch.tensor(rs.uniform(0.2, 1.0, (m, rows * cols)) * (rs.uniform(size=(m, rows * cols)) > 0.3))
    f = lambda x, n, a, r, s, e: bwd.shade_torch(x, n, a, r, s, cam, e, torch.tensor(Wn), torch.tensor(An), v, 2.2)[1]
    assert torch.autograd.gradcheck(f, args + (env,), eps=1e-7, atol=1e-6, rtol=1e-4)


# ------------------------------------------------------------------------------------------------ Eq.5 image loss
def test_image_loss_closed_forms_and_bruteforce():
    rs = np.random.default_rng(6)
    H, W = 24, 20
    I = rs.uniform(0, 1, (H, W, 3)); J = np.clip(I + rs.normal(0, 0.1, (H, W, 3)), 0, 1)
    w = bwd.ssim_window()
    assert abs(w.sum() - 1.0) < 1e-15 and np.allclose(w, w[::-1]) and w.argmax() == 5
    # identical images: SSIM = 1 everywhere, loss 0, gradient 0 (SSIM is at its maximum, |.| at its kink with subgradient 0)
    r = bwd.image_loss(I, I)
    assert abs(r["ssim"] - 1.0) < 1e-12 and abs(r["loss"]) < 1e-12 and np.abs(r["d_image"]).max() < 1e-9
    # constant images a, b: interior pixels have mu = a, mu^ = b, all variances 0 -> SSIM = (2ab + C1) / (a^2 + b^2 + C1)
    a, b = 0.7, 0.4
    r = bwd.image_loss(np.full((H, W, 3), a), np.full((H, W, 3), b))
    assert np.allclose(r["ssim_map"][5:-5, 5:-5], (2 * a * b + 1e-4) / (a * a + b * b + 1e-4), atol=1e-12)
    assert abs(r["l1"] - (a - b)) < 1e-15
    # brute force at a few pixels (also on the border: zero padding), written with explicit window sums
    r = bwd.image_loss(I, J, lam=0.2)
    for (y, x, c) in [(0, 0, 0), (3, 17, 1), (12, 10, 2), (23, 19, 0), (23, 0, 1)]:
        acc = np.zeros(5)
        for dy in range(-5, 6):
            for dx in range(-5, 6):
                yy, xx = y + dy, x + dx
                if 0 <= yy < H and 0 <= xx < W:
                    p, q = I[yy, xx, c], J[yy, xx, c]
                    acc += w[dy + 5] * w[dx + 5] * np.array([p, q, p * p, q * q, p * q])
        m1, m2 = acc[0], acc[1]; s1, s2, s12 = acc[2] - m1 * m1, acc[3] - m2 * m2, acc[4] - m1 * m2
        ref = ((2 * m1 * m2 + 1e-4) * (2 * s12 + 9e-4)) / ((m1 * m1 + m2 * m2 + 1e-4) * (s1 + s2 + 9e-4))
        assert abs(r["ssim_map"][y, x, c] - ref) < 1e-12
    assert abs(r["loss"] - (0.8 * np.abs(I - J).mean() + 0.2 * (1 - r["ssim_map"].mean()))) < 1e-14
    # gradient: central differences of the loss itself at a few pixels
    for (y, x, c) in [(0, 0, 0), (7, 9, 1), (23, 19, 2)]:
        Ip, Im = I.copy(), I.copy(); Ip[y, x, c] += 1e-6; Im[y, x, c] -= 1e-6
        fd = (bwd.image_loss(Ip, J)["loss"] - bwd.image_loss(Im, J)["loss"]) / 2e-6
        assert abs(fd - r["d_image"][y, x, c]) < 1e-8
    # lambda = 0: pure L1, gradient sign(I - I^) / (3 H W)
    r0 = bwd.image_loss(I, J, lam=0.0)
    assert np.allclose(r0["d_image"], np.sign(I - J) / I.size)


# ------------------------------------------------------------------------------------------------ Eq.6-9 regularisers
def test_regularisers_hand_example_and_finite_differences():
    # three vertices on a line, K_v = 2 neighbour sets written by hand; two Gaussians with K_g = 2
    alb = np.array([[0.1, 0.2, 0.3], [0.4, 0.2, 0.1], [0.9, 0.8, 0.7]]); rough = np.array([0.2, 0.5, 0.9]); spec = np.array([0.3, 0.3, 0.6])
    knn_v = np.array([[0, 1], [1, 0], [2, 1]])
    xv = np.array([[0.0, 0, 0], [1.0, 0, 0], [2.0, 0, 0]]); xg = np.array([[0.0, 3.0, 4.0], [1.0, 0.0, 0.0]]); knn_g = np.array([[0, 1], [1, 2]])
    disp = np.array([[0.0, 0.0, 0.0], [0.003, 0.004, 0.0], [0.0, 0.0, -0.01]])
    scale = np.array([[0.004, 0.005, 0.006], [0.02, 0.001, 0.0051]])
    r = bwd.regularisers(alb, rough, spec, knn_v, xg, xv, knn_g, disp, scale)
    # Eq.6 by hand: pairs (0,1), (1,0), (2,1) (self pairs give 0): albedo 0.5 + 0.5 + 1.7, roughness 0.3 + 0.3 + 0.4, specular 0 + 0 + 0.3
    assert np.isclose(r["smooth"], 2.7 + 1.0 + 0.3)
    assert np.allclose(r["d_rough"], [-2.0, 2.0 - 1.0, 1.0])             # vertex 1 appears as i once (+1) ... and as k twice
    assert np.allclose(r["d_spec"], [0.0, -1.0, 1.0])                    # equal values: slope 0 (reading A35)
    # Eq.7: |(0,3,4)| + |(-1,3,4)| + 0 + |(-1,0,0)| = 5 + sqrt(26) + 0 + 1
    assert np.isclose(r["mdist"], 5.0 + np.sqrt(26.0) + 1.0)
    assert np.allclose(r["d_gauss_pos"][0], np.array([0, 3, 4]) / 5.0 + np.array([-1, 3, 4]) / np.sqrt(26.0))
    assert np.allclose(r["d_gauss_pos"][1], [-1.0, 0.0, 0.0])            # the coincident vertex contributes no slope
    # Eq.8: 0 + 0.005 + 0.01;  Eq.9 with s0 = 0.005: 0.001 + 0.015 + 0.0001
    assert np.isclose(r["disp"], 0.015) and np.allclose(r["d_disp"], [[0, 0, 0], [0.6, 0.8, 0], [0, 0, -1.0]])
    assert np.isclose(r["scale"], 0.0161) and np.array_equal(r["d_scale"], [[0, 0, 1.0], [1.0, 0, 1.0]])
    # central differences on a seeded case without ties
    rs = np.random.default_rng(8)
    nv, ng = 30, 40
    args = [rs.uniform(0, 1, (nv, 3)), rs.uniform(0, 1, nv), rs.uniform(0, 1, nv), rs.integers(0, nv, (nv, 5)), rs.normal(size=(ng, 3)),
            rs.normal(size=(nv, 3)), rs.integers(0, nv, (ng, 3)), rs.normal(size=(nv, 3)) * 0.01, rs.uniform(0.001, 0.01, (ng, 3))]
    r = bwd.regularisers(*args)
    tot = lambda q: sum(q[k] for k in ("smooth", "mdist", "disp", "scale"))
    for ai, key in ((0, "d_albedo"), (1, "d_rough"), (2, "d_spec"), (4, "d_gauss_pos"), (7, "d_disp"), (8, "d_scale")):
        idx = tuple(rs.integers(0, s) for s in args[ai].shape)
        ap = [x.copy() if isinstance(x, np.ndarray) else x for x in args]; am = [x.copy() if isinstance(x, np.ndarray) else x for x in args]
        ap[ai][idx] += 1e-7; am[ai][idx] -= 1e-7
        fd = (tot(bwd.regularisers(*ap)) - tot(bwd.regularisers(*am))) / 2e-7
        assert abs(fd - r[key][idx]) < 1e-5 * (1 + abs(fd)), key


# ------------------------------------------------------------------------------------------------ H2 + Eq.1 backward
def test_pose_backward_forward_equals_cpp_oracle_and_gradcheck():
    inp = workloads.make(0)
    av = orc.avatar_load(inp)
    o = orc.render_frame(av, inp, stop_after="skin")
    N = len(inp["gauss_pos"])
    z3, z1, z6 = np.zeros((N, 3)), np.zeros(N), np.zeros((N, 6))
    r = bwd.pose_backward(inp, av["knn_g"], av["ubar_g"], 0, z3, z3, z6, z3, z1, z1)
    # same forward as orc_interp_attr + orc_skin + orc_gauss_cov (fp32 there, fp64 here)
    assert np.abs(r["xbar"] - o["gauss_posed"]).max() < 2e-6 and np.abs(r["nbar"] - o["gauss_normal_posed"]).max() < 2e-6
    assert np.allclose(r["cov6"], o["cov6"], rtol=2e-5, atol=1e-10) and np.abs(r["a_g"] - av["albedo_g"]).max() < 1e-6
    # gradcheck on a small random instance (6 Gaussians, 5 vertices, 3 bones)
    rs = np.random.default_rng(9)
    t = lambda a: torch.tensor(a, dtype=torch.float64, requires_grad=True)
    nv, ng, B = 5, 6, 3
    nn = rs.normal(size=(nv, 3)); nn /= np.linalg.norm(nn, axis=1, keepdims=True)
    w = rs.uniform(size=(nv, B)); w /= w.sum(1, keepdims=True)
    u = rs.uniform(0.1, 1, (ng, 3)); u /= u.sum(1, keepdims=True)
    args = (t(rs.normal(size=(ng, 3))), t(rs.normal(size=(ng, 4))), t(rs.uniform(0.01, 0.1, (ng, 3))), t(rs.normal(size=(B, 12))),
            t(rs.normal(size=(nv, 3)) * 0.01), t(nn), t(rs.uniform(size=(nv, 3))), t(rs.uniform(size=nv)), t(rs.uniform(size=nv)))
    knn = torch.tensor(rs.integers(0, nv, (ng, 3)))
    f = lambda *a: bwd.pose_torch(*a, knn, torch.tensor(u), torch.tensor(w))
    assert torch.autograd.gradcheck(f, args, eps=1e-7, atol=1e-7, rtol=1e-5)


def test_pose_backward_identity_pose_closed_forms():
    # every bone the identity: xbar = x_g + dx_g, nbar = n_g, Sigma = R diag(s^2) R^T.  Hand derivatives: d<g,xbar>/dx_g = g;
    # d<g,xbar>/d(dx_v[k]) = sum of ubar over the Gaussians that list k; with only d_cov6 xx = 1 and R = I: d/ds_x = 2 s_x
    inp = workloads.make(0)
    B = inp["bone_mats"].shape[1]
    inp = dict(inp); inp["bone_mats"] = np.tile(np.eye(3, 4, dtype=np.float32)[None, None], (1, B, 1, 1))
    inp["gauss_quat"] = np.tile(np.array([[1.0, 0, 0, 0]], np.float32), (len(inp["gauss_pos"]), 1))
    av = orc.avatar_load(inp)
    N, nv = len(inp["gauss_pos"]), len(inp["vert_pos"])
    g = np.random.default_rng(10).normal(size=(N, 3))
    z3, z1, z6 = np.zeros((N, 3)), np.zeros(N), np.zeros((N, 6))
    r = bwd.pose_backward(inp, av["knn_g"], av["ubar_g"], 0, g, z3, z6, z3, z1, z1)
    assert np.allclose(r["d_gauss_pos"], g)
    ref = np.zeros((nv, 3)); np.add.at(ref, av["knn_g"].reshape(-1), (av["ubar_g"][:, :, None] * g[:, None, :]).reshape(-1, 3))
    assert np.allclose(r["d_vert_disp"], ref, rtol=1e-5, atol=1e-6)       # the fp32 skinning weights sum to 1 within 1e-7
    c = z6.copy(); c[:, 0] = 1.0
    r = bwd.pose_backward(inp, av["knn_g"], av["ubar_g"], 0, z3, z3, c, z3, z1, z1)
    assert np.allclose(r["d_gauss_scale"][:, 0], 2 * inp["gauss_scale"][:, 0], rtol=1e-6) and np.allclose(r["d_gauss_scale"][:, 1:], 0, atol=1e-12)
    # Eq.1's transpose for a material attribute
    ga = np.random.default_rng(11).normal(size=(N, 3))
    r = bwd.pose_backward(inp, av["knn_g"], av["ubar_g"], 0, z3, z3, z6, ga, z1, z1)
    ref = np.zeros((nv, 3)); np.add.at(ref, av["knn_g"].reshape(-1), (av["ubar_g"][:, :, None] * ga[:, None, :]).reshape(-1, 3))
    assert np.allclose(r["d_vert_albedo"], ref, rtol=1e-12, atol=1e-12)
