"""Seeded synthetic geometry for the five BASELINE.json configs.

This module only *makes inputs* (meshes, skeletons, skinning weights).  It holds none of the
method's arithmetic (no skinning, no visibility, no shading, no splatting) and is the one
module both the oracle tests and the CUDA tests may import.

Stand-ins: the paper's canonical mesh is an SDF reconstruction remeshed to ~40K vertices
 skinned by SMPL.  Neither is available, so the body here is a
procedural 24-joint capsule figure with SMPL's *counts* (6,890 v / 13,776 f); no SMPL data is used.
"""
import os

import numpy as np

_BODY_CACHE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "data", "body_6890.npz")


# ----------------------------------------------------------------------------- icosphere
def icosphere(subdiv):
    """Unit icosphere: 10*4^s+2 vertices, 20*4^s faces, outward CCW winding."""
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
                  [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
                  [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    for _ in range(subdiv):
        v, f = subdivide(v, f)
        v /= np.linalg.norm(v, axis=1, keepdims=True)
    return v, f.astype(np.int32)


def subdivide(v, f):
    """1->4 midpoint subdivision. New vertex count = V + E."""
    f = np.asarray(f, dtype=np.int64)
    e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]], axis=0)
    es = np.sort(e, axis=1)
    key = es[:, 0] * (len(v) + 1) + es[:, 1]
    uniq, inv = np.unique(key, return_inverse=True)
    a = uniq // (len(v) + 1)
    b = uniq % (len(v) + 1)
    mid = 0.5 * (v[a] + v[b])
    nv = len(v)
    m = inv.reshape(3, -1).T + nv          # per face: midpoints of (01, 12, 20)
    m01, m12, m20 = m[:, 0], m[:, 1], m[:, 2]
    nf = np.concatenate([
        np.stack([f[:, 0], m01, m20], 1),
        np.stack([f[:, 1], m12, m01], 1),
        np.stack([f[:, 2], m20, m12], 1),
        np.stack([m01, m12, m20], 1)], axis=0)
    return np.concatenate([v, mid], axis=0), nf


def uv_sphere(rings, segs):
    """rings*segs+2 vertices, 2*rings*segs faces, outward CCW, z-up."""
    th = (np.arange(1, rings + 1)) * np.pi / (rings + 1)
    ph = np.arange(segs) * 2.0 * np.pi / segs
    T, P = np.meshgrid(th, ph, indexing="ij")
    body = np.stack([np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)], -1).reshape(-1, 3)
    v = np.concatenate([[[0, 0, 1.0]], body, [[0, 0, -1.0]]], axis=0)
    idx = lambda i, j: 1 + i * segs + (j % segs)
    faces = []
    south = 1 + rings * segs
    for j in range(segs):
        faces.append([0, idx(0, j), idx(0, j + 1)])
        faces.append([south, idx(rings - 1, j + 1), idx(rings - 1, j)])
    for i in range(rings - 1):
        for j in range(segs):
            a, b, c, d = idx(i, j), idx(i + 1, j), idx(i + 1, j + 1), idx(i, j + 1)
            faces.append([a, b, c])
            faces.append([a, c, d])
    return v, np.array(faces, dtype=np.int64)


# ----------------------------------------------------------------------------- body
# 24-joint humanoid tree in an "X" rest pose (z up, facing -y).  Names are descriptive only.
JOINT_NAMES = ["root", "spine1", "spine2", "spine3", "neck", "head",
               "l_collar", "l_shoulder", "l_elbow", "l_wrist", "l_hand",
               "r_collar", "r_shoulder", "r_elbow", "r_wrist", "r_hand",
               "l_hip", "l_knee", "l_ankle", "l_foot",
               "r_hip", "r_knee", "r_ankle", "r_foot"]
PARENTS = np.array([-1, 0, 1, 2, 3, 4,
                    3, 6, 7, 8, 9,
                    3, 11, 12, 13, 14,
                    0, 16, 17, 18,
                    0, 20, 21, 22], dtype=np.int32)


def body_skeleton():
    """Joint rest positions [24,3] (float64) and capsule list [(p0,p1,radius)]."""
    J = np.zeros((24, 3))
    J[0] = [0, 0, 0.95]
    J[1] = [0, 0, 1.08]
    J[2] = [0, 0, 1.20]
    J[3] = [0, 0, 1.32]
    J[4] = [0, 0, 1.47]
    J[5] = [0, 0, 1.60]
    arm_dir = np.array([0.19, 0.0, 1.43 - 1.10]); arm_dir /= np.linalg.norm(arm_dir)   # radial from CENTRE
    for s, base in ((1.0, 6), (-1.0, 11)):
        d = arm_dir * np.array([s, 1, 1])
        J[base + 0] = [0.08 * s, 0, 1.38]
        J[base + 1] = [0.19 * s, 0, 1.43]
        J[base + 2] = J[base + 1] + 0.27 * d
        J[base + 3] = J[base + 2] + 0.25 * d
        J[base + 4] = J[base + 3] + 0.08 * d
    leg_dir = np.array([0.09, 0.0, 0.90 - 1.10]); leg_dir /= np.linalg.norm(leg_dir)   # radial from CENTRE
    for s, base in ((1.0, 16), (-1.0, 20)):
        d = leg_dir * np.array([s, 1, 1])
        J[base + 0] = [0.09 * s, 0, 0.90]
        J[base + 1] = J[base + 0] + 0.40 * d
        J[base + 2] = J[base + 1] + 0.40 * d
        J[base + 3] = J[base + 2] + 0.09 * d
    caps = [(J[0], J[3], 0.150), (J[3], J[4], 0.135), (J[4], J[5], 0.060), (J[5], J[5] + [0, 0, 0.06], 0.105),
            (J[0] + [-0.07, 0, -0.03], J[0] + [0.07, 0, -0.03], 0.125)]
    for base in (6, 11):
        caps += [(J[3], J[base + 1], 0.075), (J[base + 1], J[base + 2], 0.052),
                 (J[base + 2], J[base + 3], 0.042), (J[base + 3], J[base + 4] + (J[base + 4] - J[base + 3]) * 0.6, 0.040)]
    for base in (16, 20):
        caps += [(J[base + 0], J[base + 1], 0.080), (J[base + 1], J[base + 2], 0.056),
                 (J[base + 2], J[base + 3] + (J[base + 3] - J[base + 2]) * 0.5, 0.050)]
    return J, caps


def _capsule_sdf(p, caps, smooth=0.03):
    """Smooth-min union of capsule SDFs; returns (sdf [N], gradient [N,3])."""
    acc = np.zeros(len(p))
    ds = []
    gs = []
    for (a, b, r) in caps:
        ab = b - a
        t = np.clip(((p - a) @ ab) / max(ab @ ab, 1e-12), 0.0, 1.0)
        q = a + t[:, None] * ab
        v = p - q
        n = np.linalg.norm(v, axis=1)
        ds.append(n - r)
        gs.append(v / np.maximum(n, 1e-12)[:, None])
    D = np.stack(ds, 1)
    G = np.stack(gs, 1)
    m = D.min(axis=1, keepdims=True)
    w = np.exp(-(D - m) / smooth)
    sw = w.sum(1, keepdims=True)
    sdf = (m - smooth * np.log(sw))[:, 0]
    grad = ((w / sw)[:, :, None] * G).sum(1)
    grad /= np.maximum(np.linalg.norm(grad, axis=1, keepdims=True), 1e-12)
    return sdf, grad


CENTRE = np.array([0.0, 0.0, 1.10])      # every limb axis passes through this point (star-shaped body)


def _radial_hit(d, caps):
    """Farthest exit of rays CENTRE + t*d from the (hard) union of capsules, closed form.
    A capsule is convex, so its exit is the largest of: the far root of its cylinder if that lies
    between the end planes, and the far roots of its two end spheres."""
    o = CENTRE
    best = np.full(len(d), 0.02)
    for (a, b, r) in caps:
        ba = b - a
        oa = o - a
        baba = ba @ ba
        bard = d @ ba
        baoa = ba @ oa
        rdoa = d @ oa
        oaoa = oa @ oa
        A = baba - bard * bard
        B = baba * rdoa - baoa * bard
        C = baba * oaoa - baoa * baoa - r * r * baba
        h = B * B - A * C
        ok = (h >= 0) & (A > 1e-14)
        t = (-B + np.sqrt(np.maximum(h, 0))) / np.where(ok, A, 1.0)
        y = baoa + t * bard
        ok &= (y >= 0) & (y <= baba)
        best = np.where(ok & (t > best), t, best)
        for c in (a, b):
            oc = o - c
            bb = d @ oc
            cc = oc @ oc - r * r
            hh = bb * bb - cc
            ts = -bb + np.sqrt(np.maximum(hh, 0))
            best = np.where((hh >= 0) & (ts > best), ts, best)
    return best


def _relax_radial(d, f, caps, iters, lam):
    """Vertices are ray directions d_i; positions CENTRE + r(d_i) d_i.  A 3D umbrella step, mapped back to a
    direction and re-cast, evens out the vertex spacing while the mesh stays a radial graph (no webbing)."""
    n = len(d)
    e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]], axis=0)
    e = np.concatenate([e, e[:, ::-1]], axis=0)
    deg = np.bincount(e[:, 0], minlength=n).astype(np.float64)
    t = _radial_hit(d, caps)
    for _ in range(iters):
        p = CENTRE + t[:, None] * d
        nb = np.zeros_like(p)
        np.add.at(nb, e[:, 0], p[e[:, 1]])
        q = p + lam * (nb / deg[:, None] - p) - CENTRE
        d = q / np.linalg.norm(q, axis=1, keepdims=True)
        t = _radial_hit(d, caps)
    return CENTRE + t[:, None] * d, d


def body_mesh(level=0):
    """level 0: 6,890 v / 13,776 f (84x82 UV-sphere topology); level 1: one subdivision -> 27,554 / 55,104."""
    J, caps = body_skeleton()
    if os.path.exists(_BODY_CACHE):                 # written by `python -m synth.mesh` (this file), ~13 s to rebuild
        z = np.load(_BODY_CACHE)
        v, f = z["v"].astype(np.float64), z["f"].astype(np.int64)
    else:
        d, f = uv_sphere(84, 82)
        v, d = _relax_radial(d, f, caps, iters=800, lam=0.5)
    if level >= 1:
        v, f = subdivide(v, f)
        q = v - CENTRE
        d = q / np.linalg.norm(q, axis=1, keepdims=True)
        v = CENTRE + _radial_hit(d, caps)[:, None] * d
    return v, f.astype(np.int32), J, caps


def two_nearest_joint_weights(v, J):
    """Dense [N_v, 24] weights: two nearest joints, inverse-distance normalised (config 1 text)."""
    d = np.linalg.norm(v[:, None, :] - J[None, :, :], axis=2)
    idx = np.argsort(d, axis=1, kind="stable")[:, :2]
    d0 = np.take_along_axis(d, idx[:, :1], 1)[:, 0]
    d1 = np.take_along_axis(d, idx[:, 1:2], 1)[:, 0]
    u0 = 1.0 / np.maximum(d0, 1e-6)
    u1 = 1.0 / np.maximum(d1, 1e-6)
    w0 = (u0 / (u0 + u1)).astype(np.float32)
    w = np.zeros((len(v), len(J)), dtype=np.float32)
    w[np.arange(len(v)), idx[:, 0]] = w0
    w[np.arange(len(v)), idx[:, 1]] = np.float32(1.0) - w0
    return w


def vertex_normals(v, f):
    """Area-weighted vertex normals (float64 in, unit float64 out)."""
    fn = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
    n = np.zeros_like(v)
    for k in range(3):
        np.add.at(n, f[:, k], fn)
    return n / np.maximum(np.linalg.norm(n, axis=1, keepdims=True), 1e-20)


if __name__ == "__main__":      # regenerate the cached base body (an input asset, not an expected value)
    if os.path.exists(_BODY_CACHE):
        os.remove(_BODY_CACHE)
    v, f, _, _ = body_mesh(0)
    os.makedirs(os.path.dirname(_BODY_CACHE), exist_ok=True)
    np.savez_compressed(_BODY_CACHE, v=v.astype(np.float64), f=f.astype(np.int32))
    print("wrote", _BODY_CACHE, v.shape, f.shape)
