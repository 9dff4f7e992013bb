"""Round-2 pins for the CPU oracle (oracle/): the parts VERDICT round 1 listed as "parity unpinned" -- orc_vis_gauss,
orc_shade's vis_mode 1 / texel_to_dir indirection, the blend's clamp / skip / stop rule, orc_window -- plus the
tightened depth-map pin and the A37 count.  Each expected value below is computed by hand in the comment beside it or
by an independent fp64 routine written here; nothing is taken from the CUDA path.  No GPU."""
import os

import numpy as np

from oracle import oracle as orc
from synth import mesh as smesh
from synth import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ Eq.1 applied to visibility
def test_vis_gauss_hand_example():
    # 4 vertices, 2 directions, K_v = 19, K_g = 3.  vcount[j][k] = number of lit vertices among S_v(j) after the filters.
    #           k=0  k=1
    vcount = np.array([[19, 0],      # vertex 0
                       [0, 19],      # vertex 1
                       [10, 5],      # vertex 2
                       [7, 3]], np.uint8)
    knn_g = np.array([[2, 0, 1],     # Gaussian 0: neighbours 2, 0, 1 with weights 1/2, 1/4, 1/4
                      [3, 3, 1]], np.int32)   # Gaussian 1: a repeated neighbour, weights 1/2, 1/8, 3/8
    ubar = np.array([[0.5, 0.25, 0.25], [0.5, 0.125, 0.375]], np.float32)
    vg = orc.vis_gauss(vcount, knn_g, ubar, 19)
    # v_g[k] = sum_j ubar_j * vcount[S_g[j]][k] / 19   (Eq.1 with the vertex visibility vbar = count / K_v)
    # G0,k0: (0.5*10 + 0.25*19 + 0.25*0)/19 = 9.75/19     G0,k1: (0.5*5 + 0.25*0 + 0.25*19)/19 = 7.25/19
    # G1,k0: (0.5*7 + 0.125*7 + 0.375*0)/19 = 4.375/19    G1,k1: (0.5*3 + 0.125*3 + 0.375*19)/19 = 9/19
    np.testing.assert_allclose(vg, [[9.75 / 19, 7.25 / 19], [4.375 / 19, 9.0 / 19]], rtol=1e-14)


def test_interp_quat_sign_alignment_hand_example():
    # reading A2 (the rotation r is a vertex attribute interpolated by Eq.1): q and -q are the same
    # rotation.  Three neighbours q, -q, q with weights 1/2, 1/4, 1/4 must give q back (a plain average gives q/2, and
    # aligning to the wrong reference or dropping the sign gives something else); the result is not normalised here.
    q = np.array([0.5, -0.5, 0.5, 0.5], np.float32)                    # a unit quaternion
    r = np.array([np.sqrt(0.5), 0, np.sqrt(0.5), 0], np.float32)       # another one, 60 degrees from q (dot = 0.7071 > 0)
    vq = np.stack([q, -q, q, r, -r]).astype(np.float32)
    idx = np.array([[0, 1, 2], [1, 0, 3], [3, 4, 1]], np.int32)
    ub = np.array([[0.5, 0.25, 0.25], [0.5, 0.25, 0.25], [0.5, 0.25, 0.25]], np.float32)
    out = orc.interp_quat(idx, ub, vq)
    np.testing.assert_allclose(out[0], q, rtol=1e-7)                   # q/2 + q/4 + q/4
    # reference = neighbour 0 = -q: 0.5(-q) + 0.25(-q) [q flipped] + 0.25(-r) [r.(-q) < 0: flipped]
    np.testing.assert_allclose(out[1], -0.75 * q - 0.25 * r, rtol=1e-6, atol=1e-7)
    # reference r: -r flipped to r; -q has dot(-q, r) < 0: flipped to q
    np.testing.assert_allclose(out[2], 0.75 * r + 0.25 * q, rtol=1e-6, atol=1e-7)
    # used through the pipeline: per-vertex quats that are all the same rotation (random signs) give that rotation's covariance
    M = np.eye(3, 4, dtype=np.float32).reshape(1, 12)
    sgn = np.array([1, -1, 1], np.float32)[:, None]
    out = orc.interp_quat(np.array([[0, 1, 2]], np.int32), np.array([[0.2, 0.3, 0.5]], np.float32), (sgn * q[None]).astype(np.float32))
    c_ref = orc.gauss_cov(M, q[None], np.array([[1.0, 2.0, 3.0]], np.float32))
    np.testing.assert_allclose(orc.gauss_cov(M, out, np.array([[1.0, 2.0, 3.0]], np.float32)), c_ref, rtol=1e-5, atol=1e-6)


# ------------------------------------------------------------------ Eq.2 with v_g and the texel -> direction map
def _one_texel_setup():
    R_, C_ = 8, 16
    w, A = orc.env_table(R_, C_)
    k = 2 * C_ + 3                                                       # the one bright texel
    env = np.zeros((R_, C_, 3), np.float32); env[2, 3] = [2.0, 3.0, 4.0]
    n = np.array([[0, 0, 1.0]], np.float32); x = np.zeros((1, 3), np.float32)
    cam = np.array([0, -3.0, 4.0], np.float32)
    alb = np.array([[0.5, 0.6, 0.7]], np.float32)
    rough, spec = np.array([0.4], np.float32), np.array([0.8], np.float32)
    return R_, C_, w, A, k, env, n, x, cam, alb, rough, spec


def test_shade_mode1_and_texel_to_dir_indirection():
    # Eq.2: L_o = sum_k L^k A^k R v_g[k] max(0, w_i.n).  With one bright texel k, the term's visibility
    # must be read at DIRECTION d = texel_to_dir[k], not at k.  K = 4 directions, texel k = 35 maps to d = 2.
    R_, C_, w, A, k, env, n, x, cam, alb, rough, spec = _one_texel_setup()
    K = 4
    t2d = np.zeros(R_ * C_, np.int32); t2d[:] = 1; t2d[k] = 2            # every other texel reads direction 1
    full, _ = orc.shade(x, n, alb, rough, spec, cam, env, None, 2)       # v = 1 everywhere (mode 2)
    assert full[0].min() > 0
    # mode 1: fractional visibility per direction; direction 2 carries 0.25, the others values that would be wrong
    vg = np.array([[0.9, 0.6, 0.25, 0.0]], np.float64)
    Lo, _ = orc.shade(x, n, alb, rough, spec, cam, env, t2d, 1, vg=vg, K=K)
    np.testing.assert_allclose(Lo[0], 0.25 * full[0], rtol=1e-14)        # L_o scales by v_g[d] = 0.25
    vg0 = np.array([[0.9, 0.6, 0.0, 1.0]], np.float64)                   # direction 2 dark, direction 3 (and k mod 4) lit
    Lo, _ = orc.shade(x, n, alb, rough, spec, cam, env, t2d, 1, vg=vg0, K=K)
    assert np.all(Lo == 0)
    # mode 0 (bits): bit d = 2 set, bit k % 32 = 3 clear -> lit; the reverse -> dark
    bits = np.array([[1 << 2]], np.uint32)
    Lo, _ = orc.shade(x, n, alb, rough, spec, cam, env, t2d, 0, bits=bits, K=K)
    np.testing.assert_allclose(Lo[0], full[0], rtol=1e-14)
    bits = np.array([[0xFFFFFFFF & ~(1 << 2)]], np.uint32)
    Lo, _ = orc.shade(x, n, alb, rough, spec, cam, env, t2d, 0, bits=bits, K=K)
    assert np.all(Lo == 0)
    # identity map with K = K_env: the bit of texel k itself (word k >> 5, bit k & 31)
    bits = np.zeros((1, 4), np.uint32); bits[0, k >> 5] = 1 << (k & 31)
    Lo, _ = orc.shade(x, n, alb, rough, spec, cam, env, None, 0, bits=bits, K=R_ * C_)
    np.testing.assert_allclose(Lo[0], full[0], rtol=1e-14)
    # gamma (reading A9, a convention): colour = clamp(L_o, 0, 1)^(1/2.2)
    _, cg = orc.shade(x, n, alb, rough, spec, cam, env, t2d, 1, vg=vg, K=K, gamma=2.2)
    np.testing.assert_allclose(cg[0], np.clip(0.25 * full[0], 0, 1) ** (1 / 2.2), rtol=1e-12)


# ------------------------------------------------------------------ blend rule (reading A18; PAPER.md:103 -> ref [8])
def _stack(opacities, W=16, H=16, mu=(8.5, 8.5), conic=(1.0, 0.0, 1.0)):
    n = len(opacities)
    mu2 = np.tile(np.array(mu, np.float32), (n, 1))
    co = np.zeros((n, 4), np.float32); co[:, 0], co[:, 1], co[:, 2] = conic; co[:, 3] = opacities
    vals = np.arange(n, dtype=np.uint32)
    ranges = np.array([[0, n]], np.uint32)
    return vals, ranges, mu2, co


def test_blend_alpha_clamp_at_099():
    # one Gaussian with o = 1 whose mean sits exactly on the centre of pixel (8, 8): power = 0, o exp(0) = 1 -> clamped to
    # 0.99 (3DGS convention): pixel = 0.99 c + 0.01 bg, T = 0.01, n_contrib = 1
    vals, ranges, mu2, co = _stack([1.0])
    col = np.array([[0.8, 0.4, 0.2]]); bg = np.array([0.5, 0.5, 1.0], np.float32)
    img, T, nc, fl = orc.composite(vals, ranges, mu2, co, col, bg, 16, 16)
    np.testing.assert_allclose(img[8, 8], 0.99 * col[0] + 0.01 * bg.astype(np.float64), rtol=1e-12)
    np.testing.assert_allclose(T[8, 8], 0.01, rtol=1e-12)
    assert nc[8, 8] == 1 and fl[8, 8] == 0
    # o = 0.995 also clamps; o = 0.98 does not
    for o, a in ((0.995, 0.99), (0.98, 0.98)):
        vals, ranges, mu2, co = _stack([o])
        img, T, _, _ = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
        np.testing.assert_allclose(T[8, 8], 1 - a, rtol=1e-6)            # fp32 opacity: 0.98f
    # one pixel to the right: d = (-1, 0), power = -0.5, alpha = exp(-0.5) unclamped
    vals, ranges, mu2, co = _stack([1.0])
    img, T, _, _ = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
    np.testing.assert_allclose(img[8, 9], np.exp(-0.5) * col[0], rtol=1e-12)


def test_blend_skip_and_stop_rule_hand_stack():
    # list (front to back) at pixel (8,8), all means on the pixel centre so alpha = opacity:
    #   #1 o = 0.002 -> alpha < 1/255: skipped (no colour, T unchanged)
    #   #2..#7 o = 0.95: T runs 0.05, 2.5e-3, 1.25e-4; the next one would give 6.25e-6 < 1e-4 -> it is REFUSED before it
    #   accumulates and the walk stops.  n_contrib is the 1-based list position of the last contributor = 4 (entries #2,
    #   #3, #4 contributed; #1 was skipped but counted), T_final = 1.25e-4.
    o95 = np.float32(0.95).astype(np.float64)
    ops = [0.002] + [0.95] * 6
    vals, ranges, mu2, co = _stack(ops)
    col = np.array([[9, 9, 9], [1, 0, 0], [0, 1, 0], [0, 0, 1], [5, 5, 5], [5, 5, 5], [5, 5, 5]], np.float64)
    img, T, nc, fl = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
    t1, t2, t3 = 1 - o95, (1 - o95) ** 2, (1 - o95) ** 3
    np.testing.assert_allclose(T[8, 8], t3, rtol=1e-12)
    assert abs(T[8, 8] - 1.25e-4) < 1e-9 and nc[8, 8] == 4 and fl[8, 8] == 0
    np.testing.assert_allclose(img[8, 8], [o95, o95 * t1, o95 * t2], rtol=1e-12)   # the white #5 never shows; nor does #1
    # a pixel 3 px away: alpha = 0.95 exp(-4.5) = 0.01055 >= 1/255 contributes; #1 (0.002 exp(-4.5)) is skipped
    a = o95 * np.exp(-4.5)
    np.testing.assert_allclose(T[8, 11], (1 - a) ** 6, rtol=1e-12)
    assert nc[8, 11] == 7
    # 4 px away: alpha = 0.95 exp(-8) = 3.2e-4 < 1/255: nothing contributes, T = 1, n_contrib = 0, pixel = bg
    bg = np.array([0.1, 0.2, 0.3], np.float32)
    img, T, nc, _ = orc.composite(vals, ranges, mu2, co, col, bg, 16, 16)
    assert T[8, 12] == 1.0 and nc[8, 12] == 0
    np.testing.assert_allclose(img[8, 12], bg.astype(np.float64), rtol=0, atol=0)


def test_blend_power_positive_is_skipped():
    # a (non-positive-definite) conic gives power > 0 away from the mean: 3DGS skips the entry; at the mean power = 0 counts
    vals, ranges, mu2, co = _stack([0.5, 0.5], conic=(-1.0, 0.0, -1.0))
    col = np.array([[1.0, 1.0, 1.0], [1.0, 1.0, 1.0]])
    img, T, nc, fl = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
    assert T[8, 9] == 1.0 and nc[8, 9] == 0                              # power = +0.5 -> skipped
    np.testing.assert_allclose(T[8, 8], 0.25, rtol=1e-12)                # power = 0 -> alpha = o, twice
    assert nc[8, 8] == 2


def test_blend_flag_band_is_narrow_and_catches_knife_edges():
    # reading A38: the flag marks decisions an fp32 evaluation may flip -- alpha within (16 + 4M) ulp of 1/255, T(1-alpha)
    # within its accumulated fp32 error of 1e-4 -- and nothing wider.
    op = np.float32(1.0 / 255.0)                                        # fp32(1/255) as opacity, power = 0 -> alpha on the edge
    vals, ranges, mu2, co = _stack([op])
    col = np.ones((1, 3))
    _, _, _, fl = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
    assert fl[8, 8] == 1
    for o in (np.float32(1.0 / 255.0 * (1 + 1e-5)), np.float32(1.0 / 255.0 * (1 - 1e-5))):      # 1e-5 relative away: decided
        vals, ranges, mu2, co = _stack([o])
        _, _, _, fl = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
        assert fl[8, 8] == 0
    # T(1 - alpha) on the 1e-4 edge: 0.9, 0.9, then a clamped 0.99: T = (1 - fp32(0.9))^2 * 0.01 = 1.0000005e-4, which is
    # 4.8e-7 (relative) above the threshold -- inside what two fp32 alphas of 0.9 can move (2 * 16 ulp * 0.9 / 0.1 = 3.4e-5)
    vals, ranges, mu2, co = _stack([0.9, 0.9, 1.0])
    _, T, nc, fl = orc.composite(vals, ranges, mu2, co, np.ones((3, 3)), np.zeros(3, np.float32), 16, 16)
    assert fl[8, 8] == 2 and nc[8, 8] == 3 and abs(T[8, 8] - 1.0000005e-4) < 1e-10          # bit 1: the stopping rule
    vals, ranges, mu2, co = _stack([0.9, 0.9, 0.985])                    # T = 1.5e-4: clearly above
    _, T, _, fl = orc.composite(vals, ranges, mu2, co, np.ones((3, 3)), np.zeros(3, np.float32), 16, 16)
    assert fl[8, 8] == 0
    # the sign of power: a (degenerate) conic a = c = 1, b = -(1 - 2^-24) three pixels off the diagonal: the terms cancel to
    # -2^-24 * 9 = 6e-8 * M / 2 -- inside 8 U M; with b = -0.99 the sum is decided
    for b, want in ((-np.float32(1.0 - 2.0 ** -24), 4), (np.float32(-0.99), 0)):
        vals, ranges, mu2, co = _stack([0.5])
        mu2 = mu2.copy(); mu2[0] = (8.5 + 3.0, 8.5 + 3.0)
        co = co.copy(); co[0, :3] = (1.0, b, 1.0)
        _, _, _, fl = orc.composite(vals, ranges, mu2, co, col, np.zeros(3, np.float32), 16, 16)
        assert (fl[8, 8] & 4) == want, (b, fl[8, 8])
    # on a real frame the band flags next to nothing (the round-1 band flagged 12 px at config 0 and 0.6 % at config 1)
    inp = workloads.make(0)
    o = orc.render_frame(orc.avatar_load(inp), inp, vis_mode=0)
    assert (o["flags"] != 0).mean() <= 1e-3


# ------------------------------------------------------------------ window (reading A13)
def test_window_of_a_box_by_hand():
    # corners (0,0,0) and (2,4,4) plus interior points: centre (1,2,2); diagonal (2,4,4) has length 6;
    # r = (0.5 * 6) * (1 + 1/64) = 3.046875 (exactly representable)
    x = np.array([[0, 0, 0], [2, 4, 4], [1, 1, 1], [0.5, 3.5, 2.0], [2, 0, 4]], np.float32)
    c, r = orc.window(x)
    assert c.tolist() == [1.0, 2.0, 2.0] and float(r) == 3.046875
    # a translated copy moves the centre only; a single point has r = 1 (degenerate rule)
    c2, r2 = orc.window(x + np.float32(8.0))
    assert c2.tolist() == [9.0, 10.0, 10.0] and float(r2) == 3.046875
    c3, r3 = orc.window(np.array([[1, 2, 3]], np.float32))
    assert c3.tolist() == [1.0, 2.0, 3.0] and float(r3) == 1.0
    # every point of the set projects inside the map for any direction: |u.(x-c)| <= r / 1.015625
    d = np.linalg.norm(x - c, axis=1)
    assert d.max() <= r / 1.015625 + 1e-6


# ------------------------------------------------------------------ depth maps (SURVEY 8(c) pins table)
def _edge_distance_px(P, f, qx, qy):
    """min distance (pixels) from each sample (qx,qy) to any triangle edge of the projected mesh P [nv,2]."""
    best = np.full(len(qx), np.inf)
    for t in f:
        for a, b in ((0, 1), (1, 2), (2, 0)):
            p0, p1 = P[t[a]], P[t[b]]
            e = p1 - p0; L2 = e @ e
            if L2 == 0:
                continue
            s = np.clip(((qx - p0[0]) * e[0] + (qy - p0[1]) * e[1]) / L2, 0, 1)
            dd = np.hypot(qx - (p0[0] + s * e[0]), qy - (p0[1] + s * e[1]))
            best = np.minimum(best, dd)
    return best


def _nearest_hit_fp64(P, Z, f, qx, qy):
    """fp64 nearest hit at samples (qx,qy) over triangles with projected corners P [nv,2] and depths Z [nv]: barycentric
    plane interpolation; returns (z or inf, |grad z| per pixel of the winning triangle)."""
    zbest = np.full(len(qx), np.inf); slope = np.zeros(len(qx))
    for t in f:
        p0, p1, p2 = P[t[0]], P[t[1]], P[t[2]]
        den = (p1[0] - p0[0]) * (p2[1] - p0[1]) - (p1[1] - p0[1]) * (p2[0] - p0[0])
        if den == 0:
            continue
        l1 = ((qx - p0[0]) * (p2[1] - p0[1]) - (qy - p0[1]) * (p2[0] - p0[0])) / den
        l2 = ((p1[0] - p0[0]) * (qy - p0[1]) - (p1[1] - p0[1]) * (qx - p0[0])) / den
        inside = (l1 >= 0) & (l2 >= 0) & (l1 + l2 <= 1)
        z = Z[t[0]] + l1 * (Z[t[1]] - Z[t[0]]) + l2 * (Z[t[2]] - Z[t[0]])
        gx = ((Z[t[1]] - Z[t[0]]) * (p2[1] - p0[1]) - (Z[t[2]] - Z[t[0]]) * (p1[1] - p0[1])) / den
        gy = (-(Z[t[1]] - Z[t[0]]) * (p2[0] - p0[0]) + (Z[t[2]] - Z[t[0]]) * (p1[0] - p0[0])) / den
        upd = inside & (z < zbest)
        zbest[upd] = z[upd]; slope[upd] = np.hypot(gx, gy)
    return zbest, slope


def test_depth_map_matches_fp64_raycast_to_1e5_away_from_edges():
    # SURVEY.md:430 "1e-5 rel ... coverage agrees except exact-edge hits".  128^2 maps of an 80-triangle ellipsoid from four
    # directions.  Independent fp64 routine: project the vertices (frame from orc.light_frames, window from the hand-pinned
    # orc_window), then at every pixel centre further than 1/128 px from every projected edge take the nearest hit by
    # barycentric plane interpolation over ALL triangles containing the sample.  There
    #  (i)  coverage agrees EXACTLY;
    #  (ii) against the true (unsnapped) geometry the depth agrees to 1e-5 + what the 1/256 px vertex snap of SURVEY 8(c)
    #       step 4 can move it (|grad z| / 256) -- a half-texel offset would be 128 times that;
    #  (iii) against the same geometry with the vertices snapped to 1/256 px in fp64 the depth agrees to 1e-5 outright.
    v, f = smesh.icosphere(1)
    v = (v * np.array([1.0, 0.7, 0.5]) + np.array([0.1, -0.2, 0.3])).astype(np.float32)
    dirs = workloads.latlong_dirs(2, 4)[[0, 3, 5, 6]]
    R = 128
    c, r = orc.window(v)
    zmap, ids = orc.vis_raster(v, f, dirs, R, c, r)
    fr = orc.light_frames(dirs).astype(np.float64)
    vd = v.astype(np.float64) - c.astype(np.float64)
    rr = float(r)
    jj, ii = np.meshgrid(np.arange(R), np.arange(R), indexing="ij")
    qx = (ii.reshape(-1) + 0.5); qy = (jj.reshape(-1) + 0.5)
    checked = 0
    for k in range(len(dirs)):
        u, vv, w = fr[k, :3], fr[k, 3:6], fr[k, 6:]
        P = np.stack([(vd @ u / rr * 0.5 + 0.5) * R, (vd @ vv / rr * 0.5 + 0.5) * R], 1)     # pixel coordinates
        Z = (rr - vd @ w) / (2 * rr)                                                          # 0 = nearest the light
        far = _edge_distance_px(P, f, qx, qy) > 1.0 / 128.0
        assert far.mean() > 0.9
        got = zmap[k].reshape(-1)
        cov = got != 0xFFFFFFFF
        gotz = got.view(np.float32).astype(np.float64)
        ztrue, slope = _nearest_hit_fp64(P, Z, f, qx, qy)
        hit = np.isfinite(ztrue)
        assert np.array_equal(cov[far], hit[far])                                           # (i)
        sel = far & hit
        err = np.abs(gotz[sel] - ztrue[sel])
        assert np.all(err <= 1e-5 + slope[sel] / 256.0), float(err.max())                   # (ii)
        zsnap, _ = _nearest_hit_fp64(np.rint(P * 256.0) / 256.0, Z, f, qx, qy)
        assert np.array_equal(np.isfinite(zsnap)[far], cov[far])
        assert np.abs(gotz[sel] - zsnap[sel]).max() <= 1e-5                                 # (iii)
        checked += int(sel.sum())
    assert checked > 8000


def test_depth_map_half_texel_and_axis_conventions():
    # one axis-aligned right triangle seen along -z (light at +z): hand-checkable coverage.  Window: c = (0,0,0), r = 2.
    # u = normalize(x^ x w) for |w_z| > 0.999 = (0,-1,0)... whatever the frame is, pixel (i,j) must be covered iff the
    # point c + ((i+1/2)/R*2-1) r u + ((j+1/2)/R*2-1) r v lies in the triangle -- a half-texel offset or a swapped axis fails.
    tri = np.array([[-1.0, -1.0, 0.5], [1.5, -1.0, 0.5], [-1.0, 1.0, 0.5]], np.float32)
    f = np.array([[0, 1, 2]], np.int32)
    w = np.array([[0.0, 0.0, 1.0]], np.float32)
    c = np.zeros(3, np.float32); r = np.float32(2.0); R = 16
    zmap, ids = orc.vis_raster(tri, f, w, R, c, r)
    fr = orc.light_frames(w)[0].astype(np.float64); u, v = fr[:3], fr[3:6]
    exp = np.zeros((R, R), bool)
    for j in range(R):
        for i in range(R):
            p = ((i + 0.5) / R * 2 - 1) * 2.0 * u + ((j + 0.5) / R * 2 - 1) * 2.0 * v
            x, y = p[0], p[1]                                              # inside: x >= -1, y >= -1, (x+1)/2.5 + (y+1)/2 <= 1
            exp[j, i] = (x >= -1) and (y >= -1) and ((x + 1) / 2.5 + (y + 1) / 2.0 <= 1)
    assert np.array_equal(zmap[0] != 0xFFFFFFFF, exp) and exp.sum() > 20
    # depth: z = (r - w.(x - c)) / (2r) = (2 - 0.5)/4 = 0.375 everywhere on the triangle
    np.testing.assert_allclose(zmap[0][exp].view(np.float32), 0.375, atol=1e-6)
    assert np.all(ids[0][exp] == 0) and np.all(ids[0][~exp] == -1)


# ------------------------------------------------------------------ reading A37: the two restatements, as numbers
def test_a37_fused_vs_plain_projection_counts():
    # oracle/a37_projection_forms.py runs the oracle in the fused form (current) and in the spelled-out form of
    # SURVEY.md:371-381 and counts what differs; the stored line for config 0 is reproduced here (config 1 takes a minute:
    # `python -m oracle.a37_projection_forms`).  The two forms never disagree on coverage; depth differs by fp32 rounding.
    from oracle import a37_projection_forms as a37
    r = a37.count(0)
    rows = [l.split() for l in open(os.path.join(GOLD, "a37_projection_forms.txt")) if l.strip() and not l.startswith("#")]
    g0 = [x for x in rows if x[0] == "0"][0]
    assert [r["texels"], r["covered"], r["coverage_differs"], r["depth_bits_differ"], r["id_differs"]] == [int(x) for x in g0[1:6]]
    assert r["vis_bits_differ"] == int(g0[8]) and r["coverage_differs"] == 0
    assert r["max_abs_depth_diff"] < 2e-7                                  # one or two fp32 ulps of a depth in [0,1]
    g1 = [x for x in rows if x[0] == "1"][0]
    assert int(g1[3]) == 0 and int(g1[8]) <= 1e-6 * int(g1[7])            # config 1: same coverage, < 1e-6 of the bits move


# ------------------------------------------------------------------ reading A40: vertex normals from the geometry
def test_vertex_normals_closed_forms_and_hand_example():
    # (1) regular octahedron, faces counter-clockwise seen from outside: by symmetry the area-weighted sum at +e_i is
    # (s, 0, 0) with the other components cancelling EXACTLY, so the normal is the vertex position itself
    v = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], np.float32)
    f = np.array([[0, 2, 4], [2, 1, 4], [1, 3, 4], [3, 0, 4], [2, 0, 5], [1, 2, 5], [3, 1, 5], [0, 3, 5]], np.int32)
    assert np.array_equal(orc.vertex_normals(v, f), v)
    # (2) winding decides the sign
    assert np.array_equal(orc.vertex_normals(v, f[:, [0, 2, 1]]), -v)
    # (3) area weighting, by hand.  O=(0,0,0) A=(2,0,0) B=(0,2,0) C=(0,0,1) and an isolated vertex D.
    #   face (O,A,B): (A-O) x (B-O) = (2,0,0) x (0,2,0) = (0,0,4)      (area 2)
    #   face (O,C,A): (C-O) x (A-O) = (0,0,1) x (2,0,0) = (0,2,0)      (area 1)
    #   O and A touch both: (0,2,4)/sqrt(20);  B only the first: (0,0,1);  C only the second: (0,1,0);  D: no face, stays 0.
    #   An unweighted mean of the two face normals would give (0,1,1)/sqrt(2) at O instead.
    v = np.array([[0, 0, 0], [2, 0, 0], [0, 2, 0], [0, 0, 1], [5, 5, 5]], np.float32)
    f = np.array([[0, 1, 2], [0, 3, 1]], np.int32)
    n = orc.vertex_normals(v, f).astype(np.float64)
    s5 = np.sqrt(5.0)
    exp = np.array([[0, 1 / s5, 2 / s5], [0, 1 / s5, 2 / s5], [0, 0, 1], [0, 1, 0], [0, 0, 0]])
    np.testing.assert_allclose(n, exp, atol=1e-7)
    # (4) a flat grid in the plane z = 3 x (not axis-aligned): every vertex normal is (-3,0,1)/sqrt(10)
    gx, gy = np.meshgrid(np.arange(5, dtype=np.float64), np.arange(4, dtype=np.float64))
    v = np.stack([gx.ravel(), gy.ravel(), 3.0 * gx.ravel()], 1).astype(np.float32)
    idx = lambda i, j: j * 5 + i
    f = np.array([t for j in range(3) for i in range(4) for t in ([idx(i, j), idx(i + 1, j), idx(i + 1, j + 1)],
                                                                 [idx(i, j), idx(i + 1, j + 1), idx(i, j + 1)])], np.int32)
    np.testing.assert_allclose(orc.vertex_normals(v, f), np.tile(np.array([-3.0, 0.0, 1.0]) / np.sqrt(10.0), (20, 1)), atol=2e-7)


def test_vertex_normals_against_fp64_on_the_body_mesh():
    # the synthetic body: the fp32 fixed-order sum agrees with an fp64 accumulation (numpy, written independently in the input
    # generator) to fp32 rounding, and a frame rendered with vert_normal = None equals one rendered with these normals passed in
    inp = workloads.make(0)
    n32 = orc.vertex_normals(inp["vert_pos"], inp["faces"])
    n64 = smesh.vertex_normals(inp["vert_pos"].astype(np.float64), inp["faces"])
    assert np.abs(n32 - n64).max() < 2e-6
    np.testing.assert_allclose(np.linalg.norm(n32.astype(np.float64), axis=1), 1.0, atol=2e-7)
    a = dict(inp); a["vert_normal"] = None
    b = dict(inp); b["vert_normal"] = n32
    oa = orc.render_frame(orc.avatar_load(a), a, stop_after="skin")
    ob = orc.render_frame(orc.avatar_load(b), b, stop_after="skin")
    assert np.array_equal(oa["gauss_normal_posed"], ob["gauss_normal_posed"]) and np.array_equal(oa["vert_normal_posed"], ob["vert_normal_posed"])
