"""Oracle of the splat's backward pass ("backward of H5-H10").  TEST INFRASTRUCTURE ONLY: imported
by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs; never by the product package.

The definition: the gradient of  L = sum_p <G(p), I(p)>  (G = dL/dimage, given) where I is the forward image of H6 + H10
(defers to 3DGS [8] :338; readings A16-A21) with its discrete decisions FROZEN -- the tile
lists and their order (H7-H9), which Gaussians are culled (near plane, facing away :101, degenerate footprint), and per
(pixel, entry) the skips (power > 0, alpha < 1/255) and the stopping rule (T < 1e-4).  Written as the forward in plain
PyTorch CPU ops in fp64 and differentiated by torch.autograd (a library primitive), so a reader can check the forward
against the paper / rga_oracle.cpp by eye and the derivative is the library's.  Where alpha is clamped to 0.99 the
derivative of the clamp is 0 (reading A32: mathematics, not the 3DGS code, which lets the gradient pass).

Pins (tests/test_backward_pins.py): the forward here equals rga_oracle.cpp's orc_project / orc_composite (independent
code); finite differences THROUGH rga_oracle.cpp reproduce the gradients; hand-derived one- and two-Gaussian closed
forms; torch.autograd.gradcheck on a tiny scene.
"""
import numpy as np
import torch

F64 = torch.float64


def _t(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64))


def project_torch(x, cov6, cam):
    """H6 (EWA projection) of the Gaussians that survive culling, differentiable.  x [n,3] posed means, cov6 [n,6]
    (xx,xy,xz,yy,yz,zz).  Same formulas and order as orc_project (rga_oracle.cpp): t = R x + t_w, clamped t_x/t_z and
    t_y/t_z (1.3 x the half field of view) inside the Jacobian only, cov2D = T Sigma T^T + 0.3 I, conic = cov2D^-1,
    mu = (fx t_x / t_z + cx, fy t_y / t_z + cy).  Returns mu [n,2], conic [n,3] (a, b, c of a dx^2 + 2 b dx dy + c dy^2)."""
    R = _t(cam["R_wc"]).reshape(3, 3); tw = _t(cam["t_wc"]).reshape(3)
    fx, fy, cx, cy = float(cam["fx"]), float(cam["fy"]), float(cam["cx"]), float(cam["cy"])
    W, H = int(cam["width"]), int(cam["height"])
    t = x @ R.T + tw
    limx, limy = 1.3 * (W / (2.0 * fx)), 1.3 * (H / (2.0 * fy))
    t0, t1, t2 = t[:, 0], t[:, 1], t[:, 2]
    txz = torch.clamp(t0 / t2, -limx, limx) * t2
    tyz = torch.clamp(t1 / t2, -limy, limy) * t2
    J00, J02 = fx / t2, -(fx * txz) / (t2 * t2)
    J11, J12 = fy / t2, -(fy * tyz) / (t2 * t2)
    T0 = J00[:, None] * R[0][None, :] + J02[:, None] * R[2][None, :]
    T1 = J11[:, None] * R[1][None, :] + J12[:, None] * R[2][None, :]
    s = cov6
    S = torch.stack([torch.stack([s[:, 0], s[:, 1], s[:, 2]], 1), torch.stack([s[:, 1], s[:, 3], s[:, 4]], 1),
                     torch.stack([s[:, 2], s[:, 4], s[:, 5]], 1)], 1)                    # [n,3,3] symmetric
    V0 = torch.einsum("na,nab->nb", T0, S); V1 = torch.einsum("na,nab->nb", T1, S)
    c00 = (V0 * T0).sum(1) + 0.3; c01 = (V0 * T1).sum(1); c11 = (V1 * T1).sum(1) + 0.3
    det = c00 * c11 - c01 * c01
    conic = torch.stack([c11 / det, -c01 / det, c00 / det], 1)
    mu = torch.stack([fx * t0 / t2 + cx, fy * t1 / t2 + cy], 1)
    return mu, conic


def composite_tile(mu, conic, opac, col, ids, pxc, pyc, bg):
    """H10 for the pixels of one tile: front-to-back "over" blend of the tile's sorted list `ids` at pixel centres
    (pxc, pyc) [P].  Same rules as blend_pixel (rga_oracle.cpp): power = -1/2 (a dx^2 + c dy^2) - b dx dy with
    d = mu - pixel; skip when power > 0; alpha = min(0.99, o exp(power)); skip when alpha < 1/255; stop before the entry
    that would take T below 1e-4; C = sum c_i alpha_i T_i + T_final bg.  The skip / stop masks are computed without
    gradient (frozen decisions).  Returns C [P,3], T_final [P], n_contrib [P] (1-based index of the last contributor)."""
    P = pxc.shape[0]
    if len(ids) == 0:
        return bg[None, :].expand(P, 3).clone(), torch.ones(P, dtype=F64), torch.zeros(P, dtype=torch.int64)
    m, q, o, c = mu[ids], conic[ids], opac[ids], col[ids]
    dx = m[None, :, 0] - pxc[:, None]; dy = m[None, :, 1] - pyc[:, None]
    power = -0.5 * (q[None, :, 0] * dx * dx + q[None, :, 2] * dy * dy) - q[None, :, 1] * dx * dy
    alpha = torch.minimum(torch.full_like(power, 0.99), o[None, :] * torch.exp(torch.clamp(power, max=0.0)))
    with torch.no_grad():
        skip = (power > 0.0) | (alpha < 1.0 / 255.0)
    alpha = torch.where(skip, torch.zeros_like(alpha), alpha)
    with torch.no_grad():
        live = torch.cumprod(1.0 - alpha, 1) >= 1e-4          # monotone: false from the stopping entry on
        idx = torch.arange(1, len(ids) + 1)[None, :].expand(P, -1)
        n_contrib = torch.where(live & ~skip, idx, torch.zeros_like(idx)).max(1).values
    alpha = torch.where(live, alpha, torch.zeros_like(alpha))
    T_incl = torch.cumprod(1.0 - alpha, 1)
    T_excl = torch.cat([torch.ones(P, 1, dtype=F64), T_incl[:, :-1]], 1)
    C = ((alpha * T_excl)[:, :, None] * c[None, :, :]).sum(1) + T_incl[:, -1:] * bg[None, :]
    return C, T_incl[:, -1], n_contrib


def splat_backward(xg, cov6, col, opac, cam, bg, vals, ranges, touched, G, mu32=None, conic32=None):
    """Forward image and the gradient of L = sum(G * image).  xg [N,3] posed means, cov6 [N,6], col [N,3] splatted
    colours, opac [N] or None (= 1), vals / ranges / touched = the frozen tile lists of H7-H9 (oracle
    outputs), G [H,W,3].  Chain rule in two stages so that only one tile's graph is alive at a time: stage 1 differentiates
    the blend w.r.t. (colour, opacity, mu, conic) tile by tile; stage 2 pulls d_mu, d_conic back through the projection.
    mu32 / conic32 (optional): the fp32 projection outputs of orc_project; when given, stage 1 blends exactly those
    values (the numbers the forward pass of either side blends), so its frozen decisions are the forward oracle's own;
    stage 2 is evaluated at the fp64 point either way.
    Returns dict with image, T_final, n_contrib, d_col, d_opac, d_mu, d_conic, d_x, d_cov6 (numpy fp64; rows of culled
    Gaussians are 0)."""
    N = len(xg); W, H = int(cam["width"]), int(cam["height"]); TX, TY = (W + 15) // 16, (H + 15) // 16
    alive = np.nonzero(np.asarray(touched) > 0)[0]
    x_a = _t(np.asarray(xg)[alive]).requires_grad_(True)
    cov_a = _t(np.asarray(cov6)[alive]).requires_grad_(True)
    mu_a, conic_a = project_torch(x_a, cov_a, cam)
    mu = torch.zeros(N, 2, dtype=F64); conic = torch.zeros(N, 3, dtype=F64)
    ia = torch.as_tensor(alive)
    mu[ia] = mu_a.detach(); conic[ia] = conic_a.detach()
    if mu32 is not None:
        mu = _t(mu32).clone(); conic = _t(np.asarray(conic32)[:, :3]).clone()
    mu.requires_grad_(True); conic.requires_grad_(True)
    colt = _t(col).requires_grad_(True)
    opt = (torch.ones(N, dtype=F64) if opac is None else _t(opac)).requires_grad_(True)
    bgt = _t(bg); Gt = _t(G)
    image = np.zeros((H, W, 3)); Tf = np.ones((H, W)); nc = np.zeros((H, W), np.int64)
    vals = np.asarray(vals).astype(np.int64); ranges = np.asarray(ranges).reshape(-1, 2)
    for ty in range(TY):
        for tx in range(TX):
            t = ty * TX + tx
            ys, xs = np.meshgrid(np.arange(ty * 16, min(ty * 16 + 16, H)), np.arange(tx * 16, min(tx * 16 + 16, W)), indexing="ij")
            ys, xs = ys.reshape(-1), xs.reshape(-1)
            ids = torch.as_tensor(vals[int(ranges[t, 0]):int(ranges[t, 1])])
            C, T, n = composite_tile(mu, conic, opt, colt, ids, _t(xs + 0.5), _t(ys + 0.5), bgt)
            image[ys, xs] = C.detach().numpy(); Tf[ys, xs] = T.detach().numpy(); nc[ys, xs] = n.numpy()
            if len(ids):
                (C * Gt[ys, xs]).sum().backward()
    z = lambda v, shape: np.zeros(shape) if v.grad is None else v.grad.numpy().copy()
    d_mu, d_conic = z(mu, (N, 2)), z(conic, (N, 3))
    torch.autograd.backward([mu_a, conic_a], [_t(d_mu[alive]), _t(d_conic[alive])])
    d_x = np.zeros((N, 3)); d_cov = np.zeros((N, 6))
    if len(alive):
        d_x[alive] = x_a.grad.numpy(); d_cov[alive] = cov_a.grad.numpy()
    return {"image": image, "T_final": Tf, "n_contrib": nc, "d_col": z(colt, (N, 3)), "d_opac": z(opt, (N,)), "d_mu": d_mu,
            "d_conic": d_conic, "d_x": d_x, "d_cov6": d_cov}


# ------------------------------------------------------------------------------------------------ H5 (shading)
def texel_visibility(n_gauss, n_texels, t2d, vis_mode, bits=None, vg=None):
    """v_g[k] per (Gaussian, env texel) as a dense fp64 array, the way orc_shade reads it: mode 0 = bit texel_to_dir[k] of
    bits[g]; mode 1 = vg[g][texel_to_dir[k]]; mode 2 = 1."""
    d = np.arange(n_texels) if t2d is None else np.asarray(t2d, np.int64)
    if vis_mode == 0:
        b = np.asarray(bits).reshape(n_gauss, -1)
        return ((b[:, d >> 5] >> (d & 31).astype(np.uint32)[None, :]) & 1).astype(np.float64)
    if vis_mode == 1:
        return np.asarray(vg, np.float64)[:, d]
    return np.ones((n_gauss, n_texels))


def shade_torch(x, n, alb, rough, spec, cam_pos, env, W, A, v, gamma):
    """H5 for a block of Gaussians, differentiable: Eq.2 with the Appendix-A BRDF (Eq.12-15, :454-471),
    same formulas and rules as orc_shade / brdf (rga_oracle.cpp): w_o = normalize(cam - x); texels with w_i.n <= 0 or
    v = 0 are skipped; s = D F / (4 ((n.w_i)(1-k)+k) ((n.w_o)^+ (1-k)+k)); L_o = sum_k L_k A_k (a/pi + p s) v (w_i.n);
    colour = clamp(L_o, 0, 1)^(1/gamma), with derivative 0 at and beyond the clamp limits (reading A33).
    x, n, alb [m,3], rough, spec [m], env [ne,3], W [ne,3], A [ne], v [m,ne].  Returns L_o [m,3], colour [m,3]."""
    PI = np.pi
    wo = cam_pos[None, :] - x
    wo = wo / wo.norm(dim=1, keepdim=True)
    cs = n @ W.T                                                     # [m,ne]  w_i . n
    with torch.no_grad():
        live = (cs > 0.0) & (v != 0.0)
    h = W[None, :, :] + wo[:, None, :]
    hl = h.norm(dim=2)
    ok = hl > 0.0
    h = h / torch.where(ok, hl, torch.ones_like(hl))[:, :, None]
    nh = (n[:, None, :] * h).sum(2); oh = (wo[:, None, :] * h).sum(2)
    no = torch.clamp((n * wo).sum(1), min=0.0)[:, None]
    al2 = (rough * rough)[:, None] ** 2                              # Eq.13: alpha = gamma^2
    den = nh * nh * (al2 - 1.0) + 1.0
    D = al2 / (PI * den * den)
    F = 0.04 + 0.96 * torch.exp2((-5.55473 * oh - 6.98316) * oh)     # Eq.14
    k = ((rough + 1.0) ** 2 / 8.0)[:, None]                          # Eq.15
    s = D * F / (4.0 * (cs * (1.0 - k) + k) * (no * (1.0 - k) + k))
    s = torch.where(ok, s, torch.zeros_like(s))
    R = alb[:, None, :] / PI + spec[:, None, None] * s[:, :, None]   # Eq.12
    term = env[None, :, :] * A[None, :, None] * R * (v * cs)[:, :, None]
    Lo = torch.where(live[:, :, None], term, torch.zeros_like(term)).sum(1)
    inside = (Lo > 0.0) & (Lo < 1.0)
    col = torch.where(inside, torch.where(inside, Lo, torch.ones_like(Lo)) ** (1.0 / gamma), (Lo >= 1.0).to(F64))
    return Lo, col


def shade_backward(xg, ng, alb, rough, spec, cam_pos, env, v, gamma, d_col, block=2048):
    """Forward radiance / colour of H5 and the gradient of L = sum(d_col * colour) w.r.t. the posed position (through w_o),
    posed normal, albedo, roughness, specular of every Gaussian and the environment map.  env [rows, cols, 3]; v dense
    visibility [N, rows*cols] (texel_visibility).  Gaussians are processed in blocks (one autograd graph at a time); the
    environment gradient accumulates over blocks.  Returns numpy fp64 arrays."""
    from . import oracle as _orc
    rows, cols = env.shape[0], env.shape[1]
    Wn, An = _orc.env_table(rows, cols)
    W, A = _t(Wn), _t(An)
    envt = _t(np.asarray(env).reshape(-1, 3)).requires_grad_(True)
    cam = _t(cam_pos)
    N = len(xg)
    out = {k: np.zeros(s) for k, s in (("Lo", (N, 3)), ("color", (N, 3)), ("d_x", (N, 3)), ("d_n", (N, 3)), ("d_alb", (N, 3)),
                                      ("d_rough", (N,)), ("d_spec", (N,)))}
    for b0 in range(0, N, block):
        sl = slice(b0, min(b0 + block, N))
        leaves = [_t(np.asarray(a)[sl]).requires_grad_(True) for a in (xg, ng, alb, rough, spec)]
        Lo, col = shade_torch(*leaves, cam, envt, W, A, _t(np.asarray(v)[sl]), gamma)
        (col * _t(np.asarray(d_col)[sl])).sum().backward()
        out["Lo"][sl] = Lo.detach().numpy(); out["color"][sl] = col.detach().numpy()
        for name, leaf in zip(("d_x", "d_n", "d_alb", "d_rough", "d_spec"), leaves):
            out[name][sl] = leaf.grad.numpy()
    out["d_env"] = (np.zeros((rows * cols, 3)) if envt.grad is None else envt.grad.numpy()).reshape(rows, cols, 3)
    return out


# ------------------------------------------------------------------------------------------------ losses, Eq.5-9
def ssim_window(size=11, sigma=1.5):
    """The SSIM window of 3DGS [8] (the paper applies "the same image loss as 3DGS"): normalised 1-D
    Gaussian, outer product with itself."""
    g = np.exp(-((np.arange(size) - size // 2) ** 2) / (2.0 * sigma * sigma))
    return g / g.sum()


def image_loss(image, target, lam=0.2):
    """Eq.5: L_img = (1 - lambda) L_1 + lambda L_D-SSIM, lambda = 0.2, and dL_img/d(image) by autograd.
    Reading A34: L_1 = mean |I - I^|; L_D-SSIM = 1 - SSIM(I, I^) as in 3DGS: per channel, 11x11 Gaussian window
    (sigma 1.5), zero padding, mu = w * I, sigma^2 = w * I^2 - mu^2, sigma_12 = w * (I I^) - mu mu^, C1 = 0.01^2,
    C2 = 0.03^2, SSIM = mean over pixels and channels of (2 mu mu^ + C1)(2 sigma_12 + C2) / ((mu^2 + mu^^2 + C1)(sigma^2 + sigma^^2 + C2)).
    image, target [H,W,3].  Returns dict loss, l1, ssim (floats) and d_image [H,W,3] (fp64)."""
    import torch.nn.functional as Fn
    I = _t(image).permute(2, 0, 1)[None].clone().requires_grad_(True)        # [1,3,H,W]
    J = _t(target).permute(2, 0, 1)[None]
    w1 = _t(ssim_window())
    w = (w1[:, None] * w1[None, :])[None, None].expand(3, 1, 11, 11).contiguous()
    conv = lambda x: Fn.conv2d(x, w, padding=5, groups=3)
    mu1, mu2 = conv(I), conv(J)
    s1 = conv(I * I) - mu1 * mu1; s2 = conv(J * J) - mu2 * mu2; s12 = conv(I * J) - mu1 * mu2
    C1, C2 = 0.01 ** 2, 0.03 ** 2
    ssim_map = ((2 * mu1 * mu2 + C1) * (2 * s12 + C2)) / ((mu1 * mu1 + mu2 * mu2 + C1) * (s1 + s2 + C2))
    ssim = ssim_map.mean()
    l1 = (I - J).abs().mean()
    loss = (1.0 - lam) * l1 + lam * (1.0 - ssim)
    loss.backward()
    return {"loss": float(loss.detach()), "l1": float(l1.detach()), "ssim": float(ssim.detach()), "d_image": I.grad[0].permute(1, 2, 0).numpy().copy(),
            "ssim_map": ssim_map.detach()[0].permute(1, 2, 0).numpy().copy()}


def regularisers(vert_albedo, vert_rough, vert_spec, knn_v, gauss_pos, vert_pos, knn_g, vert_disp, gauss_scale, s0=0.005):
    """Eq.6-9, each written as its sum, with gradients by autograd (fp64):
    Eq.6 L_smooth = sum_i sum_{k in S_v^i} ||*^i - *^k||_1 over the material attributes * in {a, gamma, p};
    Eq.7 L_mdist  = sum_i sum_{k in S_g^i} ||x_g^i - x^k||_2;   Eq.8 L_disp = sum_i ||dx^i||_2;
    Eq.9 L_scale  = sum_i max(0, s_g^i - s_0) summed over the three scale components, s_0 = 0.005.
    Reading A35: the 1-norm's slope at 0 and the 2-norm's slope at the origin are taken as 0; max(0, .) has slope 0 at 0.
    Returns dict of the four losses and d_albedo [N_v,3], d_rough [N_v], d_spec [N_v], d_gauss_pos [N_g,3], d_disp [N_v,3],
    d_scale [N_g,3]."""
    a = _t(vert_albedo).requires_grad_(True); r = _t(vert_rough).requires_grad_(True); p = _t(vert_spec).requires_grad_(True)
    xg = _t(gauss_pos).requires_grad_(True); dx = _t(vert_disp).requires_grad_(True); s = _t(gauss_scale).requires_grad_(True)
    xv = _t(vert_pos)
    kv = torch.as_tensor(np.asarray(knn_v).astype(np.int64)); kg = torch.as_tensor(np.asarray(knn_g).astype(np.int64))
    smooth = (a[:, None, :] - a[kv]).abs().sum() + (r[:, None] - r[kv]).abs().sum() + (p[:, None] - p[kv]).abs().sum()
    d = xg[:, None, :] - xv[kg]
    n2 = (d * d).sum(2)
    mdist = torch.where(n2 > 0, torch.where(n2 > 0, n2, torch.ones_like(n2)).sqrt(), torch.zeros_like(n2)).sum()
    m2 = (dx * dx).sum(1)
    disp = torch.where(m2 > 0, torch.where(m2 > 0, m2, torch.ones_like(m2)).sqrt(), torch.zeros_like(m2)).sum()
    scale = torch.where(s > s0, s - s0, torch.zeros_like(s)).sum()      # slope 0 at s = s_0 (torch.clamp would pass 1 there)
    (smooth + mdist + disp + scale).backward()                           # the four terms share no parameter
    return {"smooth": float(smooth.detach()), "mdist": float(mdist.detach()), "disp": float(disp.detach()), "scale": float(scale.detach()),
            "d_albedo": a.grad.numpy(), "d_rough": r.grad.numpy(), "d_spec": p.grad.numpy(), "d_gauss_pos": xg.grad.numpy(),
            "d_disp": dx.grad.numpy(), "d_scale": s.grad.numpy()}


# ------------------------------------------------------------------------------------------------ H2 + Eq.1 (canonical -> posed)
def pose_torch(xg, quat, scale, bones, vert_disp, vert_normal, vert_albedo, vert_rough, vert_spec, knn_g, ubar, vert_skin_w):
    """Canonical Gaussians -> posed space, differentiable (fp64): Eq.1 with the frozen neighbour sets S_g and
    weights ubar for dx_g, n_g (renormalised), w_g, a_g, gamma_g, p_g; forward LBS (:95) M = sum_b w_gb G_b,
    xbar = M [x_g + dx_g; 1], nbar = normalize(M3 n_g); covariance Sigma = A A^T, A = M3 R(q / |q|) diag(s)
    (orc_skin / orc_gauss_cov / orc_interp_attr of rga_oracle.cpp, same formulas).  bones [B,12] row-major 3x4.
    Returns xbar [N,3], nbar [N,3], cov6 [N,6], a_g [N,3], gamma_g [N], p_g [N]."""
    u = ubar[:, :, None]
    interp = lambda t: (u * t[knn_g]).sum(1) if t.dim() == 2 else (ubar * t[knn_g]).sum(1)
    dx, nraw, w = interp(vert_disp), interp(vert_normal), interp(vert_skin_w)
    a_g, r_g, p_g = interp(vert_albedo), interp(vert_rough), interp(vert_spec)
    n_g = nraw / nraw.norm(dim=1, keepdim=True)
    M = (w @ bones).reshape(-1, 3, 4)
    M3, tr = M[:, :, :3], M[:, :, 3]
    p = xg + dx
    xbar = torch.einsum("nrc,nc->nr", M3, p) + tr
    t = torch.einsum("nrc,nc->nr", M3, n_g)
    nbar = t / t.norm(dim=1, keepdim=True)
    q = quat / quat.norm(dim=1, keepdim=True)
    qw, qx, qy, qz = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = torch.stack([1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy),
                     2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx),
                     2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy)], 1).reshape(-1, 3, 3)
    A = M3 @ (R * scale[:, None, :])
    S = A @ A.transpose(1, 2)
    cov6 = torch.stack([S[:, 0, 0], S[:, 0, 1], S[:, 0, 2], S[:, 1, 1], S[:, 1, 2], S[:, 2, 2]], 1)
    return xbar, nbar, cov6, a_g, r_g, p_g


def pose_backward(inp, knn_g, ubar, frame, d_mean, d_normal, d_cov6, d_alb_g, d_rough_g, d_spec_g):
    """Gradient of L = <d_mean, xbar> + <d_normal, nbar> + <d_cov6, cov6> + <d_alb_g, a_g> + <d_rough_g, gamma_g> + <d_spec_g, p_g>
    w.r.t. the canonical Gaussian position, rotation and scale, the bone transforms of the pose, and the vertex attributes
    dx, n, a, gamma, p (through Eq.1's transpose; S_g, ubar and the skinning weights are frozen).  inp: the workload dict."""
    T = lambda a: _t(a).requires_grad_(True)
    leaves = {"d_gauss_pos": T(inp["gauss_pos"]), "d_gauss_quat": T(inp["gauss_quat"]), "d_gauss_scale": T(inp["gauss_scale"]),
              "d_bones": T(np.asarray(inp["bone_mats"][frame]).reshape(-1, 12)), "d_vert_disp": T(inp["vert_disp"]),
              "d_vert_normal": T(inp["vert_normal"]), "d_vert_albedo": T(inp["vert_albedo"]), "d_vert_rough": T(inp["vert_rough"]),
              "d_vert_spec": T(inp["vert_spec"])}
    outs = pose_torch(*leaves.values(), torch.as_tensor(np.asarray(knn_g).astype(np.int64)), _t(ubar), _t(inp["vert_skin_w"]))
    cot = [d_mean, d_normal, d_cov6, d_alb_g, d_rough_g, d_spec_g]
    sum((o * _t(c)).sum() for o, c in zip(outs, cot)).backward()
    res = {k: v.grad.numpy() for k, v in leaves.items()}
    res.update({"xbar": outs[0].detach().numpy(), "nbar": outs[1].detach().numpy(), "cov6": outs[2].detach().numpy(),
                "a_g": outs[3].detach().numpy()})
    return res
