"""Seeded synthetic workloads: the five BASELINE.json configs as plain numpy arrays.

Inputs only.  No step of the method (Eq.1 interpolation, skinning, visibility, shading, splatting)
is computed here; the oracle (oracle/) and the CUDA library (paper_2407_10707_b200/) each receive
these same arrays.  Recipe and the stand-in statement: DESIGN.md "Synthetic inputs".
"""
import functools

import numpy as np

from . import mesh as _mesh

CONFIG_NAMES = ["tiny", "smpl", "highres", "anim", "stress"]

#            mesh      N_g        env(R,C)  K_vis(Rd,Cd) R_v  W     H     frames n_env opacity
_CFG = {
    0: dict(mesh="ico", n_gauss=2_000, env=(8, 16), dirs=(2, 8), vis_res=64, width=64, height=64,
            frames=1, n_env=1, op=(0.1, 0.99), env_kind="uniform"),
    1: dict(mesh="body0", n_gauss=100_000, env=(16, 32), dirs=(16, 32), vis_res=128, width=512, height=512,
            frames=1, n_env=1, op=(0.1, 0.99), env_kind="lognormal"),
    2: dict(mesh="body1", n_gauss=300_000, env=(32, 64), dirs=(16, 32), vis_res=256, width=1024, height=1024,
            frames=1, n_env=1, op=(0.1, 0.99), env_kind="lognormal"),
    3: dict(mesh="body0", n_gauss=100_000, env=(16, 32), dirs=(16, 32), vis_res=128, width=512, height=512,
            frames=64, n_env=4, op=(0.1, 0.99), env_kind="lognormal"),
    4: dict(mesh="body1", n_gauss=1_000_000, env=(32, 64), dirs=(16, 64), vis_res=256, width=1920, height=1080,
            frames=1, n_env=1, op=(0.5, 0.99), env_kind="lognormal"),
}


def _rng(seed, stream):
    return np.random.default_rng(np.random.SeedSequence([seed, stream]))


def _rodrigues(axis, angle):
    axis = axis / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + np.sin(angle) * K + (1 - np.cos(angle)) * (K @ K)


def bone_matrices(J, parents, rot):
    """Host-side forward kinematics in float64: G_b = posed_global_b * inverse_bind_b, returned [B,12] fp32
    (row-major 3x4).  The boundary takes bone matrices, not SMPL theta (reading A5)."""
    B = len(J)
    G = np.zeros((B, 4, 4))
    for b in range(B):
        L = np.eye(4)
        L[:3, :3] = rot[b]
        pj = J[parents[b]] if parents[b] >= 0 else np.zeros(3)
        L[:3, 3] = J[b] - pj
        G[b] = L if parents[b] < 0 else G[parents[b]] @ L
    out = np.zeros((B, 12), dtype=np.float32)
    for b in range(B):
        inv_bind = np.eye(4)
        inv_bind[:3, 3] = -J[b]
        out[b] = (G[b] @ inv_bind)[:3, :].reshape(12).astype(np.float32)
    return out


def latlong_dirs(rows, cols):
    """Unit vectors at the texel centres of a z-up lat-long grid, pointing toward the light (fp32, [rows*cols,3])."""
    th = (np.arange(rows) + 0.5) * np.pi / rows
    ph = (np.arange(cols) + 0.5) * 2.0 * np.pi / cols
    T, P = np.meshgrid(th, ph, indexing="ij")
    d = np.stack([np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)], -1).reshape(-1, 3)
    d = d.astype(np.float32)
    d /= np.linalg.norm(d.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
    return np.ascontiguousarray(d, dtype=np.float32)


def texel_to_dir(env_rc, dir_rc):
    """Integer block map from env texel (i,j) to the coarser direction grid (reading A12)."""
    R, C = env_rc
    Rd, Cd = dir_rc
    i = np.arange(R)[:, None] * Rd // R
    j = np.arange(C)[None, :] * Cd // C
    return np.ascontiguousarray((i * Cd + j).reshape(-1), dtype=np.int32)


def _morton_order(p):
    lo, hi = p.min(0), p.max(0)
    q = np.clip(((p - lo) / np.maximum(hi - lo, 1e-12) * 1023.0), 0, 1023).astype(np.uint64)

    def spread(x):
        x = (x | (x << np.uint64(16))) & np.uint64(0x030000FF)
        x = (x | (x << np.uint64(8))) & np.uint64(0x0300F00F)
        x = (x | (x << np.uint64(4))) & np.uint64(0x030C30C3)
        x = (x | (x << np.uint64(2))) & np.uint64(0x09249249)
        return x
    code = spread(q[:, 0]) | (spread(q[:, 1]) << np.uint64(1)) | (spread(q[:, 2]) << np.uint64(2))
    return np.argsort(code, kind="stable")


@functools.lru_cache(maxsize=8)
def _base_mesh(kind):
    if kind == "ico":
        v, f = _mesh.icosphere(3)
        J = np.array([[0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
        parents = np.array([-1, 0], dtype=np.int32)
        z = np.clip((v[:, 2] + 0.5) / 1.0, 0.0, 1.0)
        w2 = z * z * (3.0 - 2.0 * z)
        w = np.stack([1.0 - w2.astype(np.float32), w2.astype(np.float32)], 1).astype(np.float32)
        return v, f, J, parents, w
    v, f, J, _ = _mesh.body_mesh(0 if kind == "body0" else 1)
    return v, f, J, _mesh.PARENTS.copy(), _mesh.two_nearest_joint_weights(v, J)


def make(cfg_id, seed=None, n_gauss=None, morton=False):
    """Return a dict of contiguous numpy arrays for config `cfg_id` (0..4).  `n_gauss` overrides the count
    (used by tests to shrink a config while keeping its structure).  Gaussians come in the order they were drawn
    ("random surface points", BASELINE.json); `morton=True` stores them in Morton order of their canonical position
    instead (bench.py reports that variant beside the metric)."""
    c = dict(_CFG[cfg_id])
    seed = cfg_id if seed is None else seed
    if n_gauss is not None:
        c["n_gauss"] = int(n_gauss)
    v, f, J, parents, w = _base_mesh(c["mesh"])
    B = len(J)
    out = dict(cfg_id=cfg_id, name=CONFIG_NAMES[cfg_id], n_bones=B)
    out["vert_pos"] = np.ascontiguousarray(v, dtype=np.float32)
    out["faces"] = np.ascontiguousarray(f, dtype=np.int32)
    out["vert_normal"] = np.ascontiguousarray(_mesh.vertex_normals(v, f), dtype=np.float32)
    out["vert_skin_w"] = np.ascontiguousarray(w, dtype=np.float32)
    out["vert_disp"] = np.zeros_like(out["vert_pos"])          # A4: static average displacement, 0 in the configs
    r = _rng(seed, 1)
    nv = len(v)
    out["vert_albedo"] = r.uniform(0.0, 1.0, (nv, 3)).astype(np.float32)
    out["vert_rough"] = r.uniform(0.1, 1.0, nv).astype(np.float32)
    out["vert_spec"] = r.uniform(0.0, 1.0, nv).astype(np.float32)

    # Gaussians: triangle ~ area, uniform barycentric, + N(0, 0.005) along the face normal
    r = _rng(seed, 2)
    ng = c["n_gauss"]
    fn = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
    area = 0.5 * np.linalg.norm(fn, axis=1)
    tri = r.choice(len(f), size=ng, p=area / area.sum())
    u1 = np.sqrt(r.uniform(0, 1, ng)); u2 = r.uniform(0, 1, ng)
    b0, b1, b2 = 1 - u1, u1 * (1 - u2), u1 * u2
    p = b0[:, None] * v[f[tri, 0]] + b1[:, None] * v[f[tri, 1]] + b2[:, None] * v[f[tri, 2]]
    nrm = fn[tri] / np.maximum(np.linalg.norm(fn[tri], axis=1, keepdims=True), 1e-20)
    p = p + r.normal(0.0, 0.005, ng)[:, None] * nrm
    scale = np.exp(r.uniform(np.log(1e-3), np.log(1e-2), (ng, 3)))
    quat = r.normal(0, 1, (ng, 4)); quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    opac = r.uniform(c["op"][0], c["op"][1], ng)
    if morton:
        o = _morton_order(p)
        p, scale, quat, opac = p[o], scale[o], quat[o], opac[o]
    out["gauss_pos"] = np.ascontiguousarray(p, dtype=np.float32)
    out["gauss_scale"] = np.ascontiguousarray(scale, dtype=np.float32)
    out["gauss_quat"] = np.ascontiguousarray(quat, dtype=np.float32)     # (w,x,y,z)
    out["gauss_opacity"] = np.ascontiguousarray(opac, dtype=np.float32)

    # poses -> bone matrices [frames, B, 12]
    r = _rng(seed, 3)
    nfr = c["frames"]
    mats = np.zeros((nfr, B, 12), dtype=np.float32)
    if c["mesh"] == "ico":
        rot = [np.eye(3), _rodrigues(np.array([1.0, 0, 0]), np.deg2rad(30.0))]
        mats[0] = bone_matrices(J, parents, rot)
    else:
        axes = r.normal(0, 1, (B, 3))
        if nfr == 1:
            ang = np.deg2rad(r.uniform(-30, 30, B))[None, :]
        else:
            phase = r.uniform(0, 2 * np.pi, B)
            t = np.arange(nfr)[:, None]
            ang = np.deg2rad(30.0) * np.sin(2 * np.pi * t / nfr + phase[None, :])
        for t in range(nfr):
            rot = [np.eye(3)] + [_rodrigues(axes[b], ang[t, b]) for b in range(1, B)]
            mats[t] = bone_matrices(J, parents, rot)
    out["bone_mats"] = mats

    # environment maps [n_env, R, C, 3] and which map each frame uses
    r = _rng(seed, 4)
    R, C = c["env"]
    if c["env_kind"] == "uniform":
        env = r.uniform(0.0, 2.0, (c["n_env"], R, C, 3))
    else:
        env = np.exp(r.normal(0.0, 1.0, (c["n_env"], R, C, 3)))
    out["env"] = np.ascontiguousarray(env, dtype=np.float32)
    out["env_of_frame"] = r.integers(0, c["n_env"], nfr).astype(np.int32) if c["n_env"] > 1 else np.zeros(nfr, np.int32)
    out["env_rows"], out["env_cols"] = R, C
    out["gamma"] = 2.2

    # visibility directions and the env-texel -> direction map (A12)
    Rd, Cd = c["dirs"]
    out["vis_dirs"] = latlong_dirs(Rd, Cd)
    out["texel_to_dir"] = texel_to_dir((R, C), (Rd, Cd))
    out["vis_res"] = c["vis_res"]
    out["depth_bias_texels"] = 1.0
    out["depth_bias_world"] = 0.015
    out["slope_max"] = 8.0

    # camera: vertical FoV 40 deg, looking along +y (world) at the canonical AABB centre, z up
    W, H = c["width"], c["height"]
    lo, hi = v.min(0), v.max(0)
    ctr = 0.5 * (lo + hi)
    rb = 0.5 * np.linalg.norm(hi - lo) * 1.05
    dist = rb / np.sin(np.deg2rad(20.0))
    cam_pos = ctr + np.array([0.0, -dist, 0.0])
    R_wc = np.array([[1.0, 0, 0], [0, 0, -1.0], [0, 1.0, 0]])
    t_wc = -R_wc @ cam_pos
    fy = 0.5 * H / np.tan(np.deg2rad(20.0))
    out["camera"] = dict(R_wc=R_wc.astype(np.float32).reshape(9), t_wc=t_wc.astype(np.float32),
                         fx=np.float32(fy), fy=np.float32(fy), cx=np.float32(W / 2), cy=np.float32(H / 2),
                         width=W, height=H, z_near=np.float32(0.2))
    out["cam_pos"] = cam_pos.astype(np.float32)
    out["bg"] = np.zeros(3, dtype=np.float32)
    return out


def make_random(seed):
    """A small RANDOM configuration for the randomised parity sweep (tests/test_gpu_random_configs.py): config 0 or 1 with
    500..9000 Gaussians and everything the hot path is parameterised by drawn at random -- direction grid (K not a multiple
    of 32), environment map (1..6 texels per direction), depth-map side (8..256, odd sizes), bias constants, Gaussian scale
    and opacity ranges, image size (not a multiple of the 16-pixel tile), camera position / orientation / focal lengths /
    principal point / near plane (close-ups give long tile lists), background, gamma, and in a third of the cases no vertex
    normals (the library computes them).  Returns (inputs, description).  Inputs only."""
    rs = np.random.default_rng(10_000 + seed)
    base = int(rs.choice([0, 1, 1]))
    ng = int(rs.integers(500, 9000))
    inp = make(base, seed=seed, n_gauss=ng)
    Rd, Cd = int(rs.integers(1, 7)), int(rs.integers(1, 13))
    mr, mc = int(rs.choice([1, 1, 2, 3])), int(rs.choice([1, 1, 2]))
    R, C = Rd * mr, Cd * mc
    inp["vis_dirs"] = latlong_dirs(Rd, Cd)
    inp["texel_to_dir"] = texel_to_dir((R, C), (Rd, Cd))
    env = rs.uniform(0, 2, (1, R, C, 3)) if rs.integers(0, 2) == 0 else np.exp(rs.normal(0, 1, (1, R, C, 3)))
    inp["env"] = np.ascontiguousarray(env, np.float32)
    inp["env_rows"], inp["env_cols"] = R, C
    inp["env_of_frame"] = np.zeros(len(inp["bone_mats"]), np.int32)
    inp["vis_res"] = int(rs.choice([8, 17, 33, 64, 100, 128, 129, 200, 256]))
    inp["depth_bias_texels"] = float(rs.choice([0.0, 0.5, 1.0, 2.0]))
    inp["depth_bias_world"] = float(rs.choice([0.0, 0.005, 0.015, 0.05]))
    inp["slope_max"] = float(rs.choice([1.0, 2.0, 8.0, 50.0]))
    smax = float(rs.choice([5e-3, 1e-2, 3e-2, 8e-2]))
    inp["gauss_scale"] = np.exp(rs.uniform(np.log(1e-3), np.log(smax), (ng, 3))).astype(np.float32)
    inp["gauss_opacity"] = rs.uniform(float(rs.choice([0.05, 0.3, 0.9])), 1.0, ng).astype(np.float32)
    v = inp["vert_pos"]
    lo3, hi3 = v.min(0), v.max(0)
    ctr = 0.5 * (lo3 + hi3)
    rb = 0.5 * np.linalg.norm(hi3 - lo3)
    W, H = int(rs.integers(20, 400)), int(rs.integers(20, 400))
    az, el = rs.uniform(0, 2 * np.pi), rs.uniform(-1.2, 1.2)
    dist = rb * float(rs.choice([0.6, 1.0, 2.0, 3.5]) if base == 1 else rs.choice([2.0, 3.5]))   # config 0 is a ball: stay outside
    fwd = -np.array([np.cos(el) * np.cos(az), np.cos(el) * np.sin(az), np.sin(el)])
    cam_pos = ctr - fwd * dist + rs.normal(0, 0.05, 3)
    right = np.cross(fwd, np.array([0, 0, 1.0])); right /= np.linalg.norm(right)
    R_wc = np.stack([right, np.cross(fwd, right), fwd])
    fy = 0.5 * H / np.tan(0.5 * np.deg2rad(float(rs.choice([25, 40, 70]))))
    inp["camera"] = dict(R_wc=R_wc.astype(np.float32).reshape(9), t_wc=(-R_wc @ cam_pos).astype(np.float32),
                         fx=np.float32(fy * rs.uniform(0.8, 1.2)), fy=np.float32(fy), cx=np.float32(W / 2 + rs.uniform(-5, 5)),
                         cy=np.float32(H / 2 + rs.uniform(-5, 5)), width=W, height=H, z_near=np.float32(rs.choice([0.05, 0.2, 0.8])))
    inp["cam_pos"] = cam_pos.astype(np.float32)
    inp["bg"] = rs.uniform(0, 1, 3).astype(np.float32)
    inp["gamma"] = float(rs.choice([1.0, 2.2]))
    if rs.uniform() < 0.3:
        inp["vert_normal"] = None
    desc = dict(seed=seed, base=base, n_gauss=ng, dirs=(Rd, Cd), env=(R, C), vis_res=inp["vis_res"], image=(W, H),
                dist=round(float(dist), 2), scale_max=smax, normals=inp["vert_normal"] is not None)
    return inp, desc


def make_disp_mlp(seed=0, n_freq=64, n_pose=72, width=256, n_hidden=4, rff_sigma=1.0, out_scale=0.01):
    """Random weights of the displacement network d(x, theta): the trained weights are not
    available, so these are seeded stand-ins with the architecture of DESIGN.md readings A26-A28 (He-initialised hidden
    layers, a head scaled so that |dx| is about a centimetre) and a random pose vector theta.  Inputs only."""
    r = _rng(seed, 7)
    d_in = 2 * n_freq + n_pose
    he = lambda fan_in, shape: (r.standard_normal(shape) * np.sqrt(2.0 / fan_in)).astype(np.float32)
    return dict(
        n_freq=n_freq, n_pose=n_pose,
        rff=(rff_sigma * r.standard_normal((n_freq, 3))).astype(np.float32),
        W1=he(d_in, (width, d_in)), b1=(0.1 * r.standard_normal(width)).astype(np.float32),
        Wh=he(width, (n_hidden - 1, width, width)), bh=(0.1 * r.standard_normal((n_hidden - 1, width))).astype(np.float32),
        Wo=(out_scale * he(width, (3, width))).astype(np.float32), bo=(0.001 * r.standard_normal(3)).astype(np.float32),
        theta=np.deg2rad(r.uniform(-30.0, 30.0, n_pose)).astype(np.float32))


def make_image_cotangent(seed, width, height):
    """dL/dimage for the backward pass: a seeded standard-normal field [height, width, 3] (fp32).  An input of both the
    oracle and the library; the loss that would produce it (Eq.5) is not part of this module."""
    return np.random.default_rng(1000 + seed).normal(size=(height, width, 3)).astype(np.float32)


def make_color_cotangent(seed, n_gauss):
    """dL/dcolour per Gaussian for the backward of the shading step: seeded standard normal [n_gauss, 3] (fp32)."""
    return np.random.default_rng(2000 + seed).normal(size=(n_gauss, 3)).astype(np.float32)


def make_image_pair(seed, width, height):
    """(rendered, target) stand-ins for the image loss: a smooth seeded random field in [0,1] (sum of a few low-frequency
    cosines per channel) as target, and the same plus small-scale noise, clipped, as the rendered image.  fp32 [H,W,3]."""
    rs = np.random.default_rng(3000 + seed)
    y, x = np.meshgrid(np.arange(height) / max(height, 1), np.arange(width) / max(width, 1), indexing="ij")
    tgt = np.zeros((height, width, 3))
    for c in range(3):
        for _ in range(6):
            fx, fy, ph = rs.uniform(0.5, 6.0), rs.uniform(0.5, 6.0), rs.uniform(0, 2 * np.pi)
            tgt[:, :, c] += rs.uniform(0.05, 0.2) * np.cos(2 * np.pi * (fx * x + fy * y) + ph)
    tgt = np.clip(0.5 + tgt, 0.0, 1.0)
    img = np.clip(tgt + rs.normal(0.0, 0.05, tgt.shape), 0.0, 1.0)
    img[: height // 4, : width // 4] = 0.0                                # a black corner: zero-variance windows on one side
    return img.astype(np.float32), tgt.astype(np.float32)


def make_cotangent(seed, shape):
    """A seeded standard-normal cotangent (fp32) of any shape, for the backward tests and benches."""
    return np.random.default_rng(4000 + seed).normal(size=shape).astype(np.float32)
