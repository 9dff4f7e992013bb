"""Thin ctypes binding of librga.so (include/rga.h).  Argument marshalling only: every step of the path runs in the
CUDA kernels.  Torch supplies device memory and the current stream.  Nothing here imports or calls oracle/."""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "librga.so")

RGA_OK, RGA_ERR_INVALID_ARG, RGA_ERR_CUDA, RGA_ERR_OOM, RGA_ERR_STATE, RGA_ERR_CAPACITY = range(6)

# rga_buffer_id -> (name, numpy dtype, trailing shape or None)
BUF = dict(KNN_G=0, UBAR_G=1, KNN_V=2, GAUSS_STATIC=3, GAUSS_SKIN_W=4, VERT_POSED=5, VERT_NORMAL_POSED=6, GAUSS_POSED=7,
           GAUSS_NORMAL_POSED=8, GAUSS_COV=9, WINDOW=10, ZMAP=11, IDMAP=12, VISBITS=13, VCOUNT=14, RADIANCE=15, COLOR=16,
           MU2D=17, DEPTH=18, CONIC_OPACITY=19, RECT=20, TOUCHED=21, NUM_DUPLICATES=22, KEYS_SORTED=23, VALS_SORTED=24,
           TILE_RANGES=25, T_FINAL=26, N_CONTRIB=27, VERT_BITS_RAW=28, VERT_DISP=29,
           DENS_DV=30, DENS_P=31, DENS_NG=32, DENS_HDR=33, SPLAT_GRAD=34, GAUSS_ORDER=35, VERT_NORMAL=36)
_BUF_DTYPE = {0: np.int32, 1: np.float32, 2: np.int32, 3: np.float32, 4: np.float32, 5: np.float32, 6: np.float32,
              7: np.float32, 8: np.float32, 9: np.float32, 10: np.float32, 11: np.uint32, 12: np.int32, 13: np.uint32,
              14: np.uint8, 15: np.float32, 16: np.float32, 17: np.float32, 18: np.float32, 19: np.float32, 20: np.int32,
              21: np.uint32, 22: np.uint32, 23: np.uint64, 24: np.uint32, 25: np.uint32, 26: np.float32, 27: np.uint32,
              28: np.uint32, 29: np.float32, 30: np.int32, 31: np.uint32, 32: np.int32, 33: np.uint64, 34: np.float32, 35: np.int32, 36: np.float32}


class RgaError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("rga status %d: %s" % (status, msg))
        self.status = status


class _Desc(C.Structure):
    _fields_ = [("n_verts", C.c_int32), ("n_faces", C.c_int32), ("n_bones", C.c_int32), ("n_gauss", C.c_int32),
                ("k_g", C.c_int32), ("k_v", C.c_int32),
                ("vert_pos", C.c_void_p), ("faces", C.c_void_p), ("vert_normal", C.c_void_p), ("vert_skin_w", C.c_void_p),
                ("vert_disp", C.c_void_p), ("vert_albedo", C.c_void_p), ("vert_rough", C.c_void_p), ("vert_spec", C.c_void_p),
                ("gauss_pos", C.c_void_p), ("gauss_quat", C.c_void_p), ("gauss_scale", C.c_void_p), ("gauss_opacity", C.c_void_p),
                ("max_width", C.c_int32), ("max_height", C.c_int32), ("max_vis_dirs", C.c_int32), ("max_vis_res", C.c_int32),
                ("max_env_texels", C.c_int32), ("max_duplicates", C.c_int64), ("vert_quat", C.c_void_p), ("vert_scale", C.c_void_p)]


class _Camera(C.Structure):
    _fields_ = [("R_wc", C.c_float * 9), ("t_wc", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float),
                ("cy", C.c_float), ("width", C.c_int32), ("height", C.c_int32), ("z_near", C.c_float)]


class _VisParams(C.Structure):
    _fields_ = [("n_dirs", C.c_int32), ("res", C.c_int32), ("mode", C.c_int32), ("dirs", C.c_void_p),
                ("depth_bias_texels", C.c_float), ("depth_bias_world", C.c_float), ("slope_max", C.c_float),
                ("keep_maps", C.c_int32), ("cull_backfaces", C.c_int32)]


class _Env(C.Structure):
    _fields_ = [("rows", C.c_int32), ("cols", C.c_int32), ("radiance", C.c_void_p), ("texel_to_dir", C.c_void_p),
                ("gamma", C.c_float), ("use_visibility", C.c_int32)]


_lib = None


def lib():
    """Load librga.so; fail loudly when it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("librga.so is missing: run `python -m paper_2407_10707_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_LIB_PATH)
        L.rga_last_error.restype = C.c_char_p
        L.rga_version.restype = C.c_char_p
        L.rga_launch_count.restype = C.c_int64
        L.rga_launch_count.argtypes = [C.c_void_p]
        L.avatar_load.argtypes = [C.POINTER(_Desc), C.c_void_p, C.POINTER(C.c_void_p)]
        L.avatar_free.argtypes = [C.c_void_p]
        L.pose_skin.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.visibility_raster.argtypes = [C.c_void_p, C.POINTER(_VisParams), C.c_void_p]
        L.shade_gaussians.argtypes = [C.c_void_p, C.POINTER(_Env), C.POINTER(C.c_float), C.c_void_p]
        L.splat_render.argtypes = [C.c_void_p, C.POINTER(_Camera), C.POINTER(C.c_float), C.c_void_p, C.c_void_p]
        L.splat_attribute.argtypes = [C.c_void_p, C.POINTER(_Camera), C.POINTER(C.c_float), C.c_int, C.c_void_p, C.c_void_p]
        L.rga_render_frame.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_VisParams), C.POINTER(_Env), C.POINTER(C.c_float),
                                       C.POINTER(_Camera), C.POINTER(C.c_float), C.c_void_p, C.c_void_p]
        L.rga_get_buffer.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
        L.rga_read_buffer.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_size_t)]
        L.rga_check.argtypes = [C.c_void_p, C.c_void_p]
        L.rga_profile_enable.argtypes = [C.c_void_p, C.c_int]
        L.rga_profile_read.argtypes = [C.c_void_p, C.c_void_p, C.c_char_p, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_int)]
        _lib = L
    return _lib


def _chk(st):
    if st != RGA_OK:
        raise RgaError(st, lib().rga_last_error().decode())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(a, dtype):
    """numpy / torch array -> contiguous CUDA tensor of `dtype` (an upload, not arithmetic)."""
    if a is None:
        return None
    t = torch.as_tensor(a) if not isinstance(a, torch.Tensor) else a
    return t.to(device="cuda", dtype=dtype).contiguous()


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def make_camera(cam):
    c = _Camera()
    c.R_wc[:] = [float(v) for v in np.asarray(cam["R_wc"], np.float32).reshape(9)]
    c.t_wc[:] = [float(v) for v in np.asarray(cam["t_wc"], np.float32).reshape(3)]
    c.fx, c.fy, c.cx, c.cy = float(cam["fx"]), float(cam["fy"]), float(cam["cx"]), float(cam["cy"])
    c.width, c.height, c.z_near = int(cam["width"]), int(cam["height"]), float(cam["z_near"])
    return c


# ----------------------------------------------------------------------------------------------- C-ABI entry points
def avatar_load(inp, max_width, max_height, max_vis_dirs, max_vis_res, max_env_texels, max_duplicates=0, k_g=3, k_v=19):
    """L0 (include/rga.h avatar_load).  `inp` holds the tables of rga_avatar_desc as numpy or torch arrays."""
    if not torch.cuda.is_available():
        raise RgaError(RGA_ERR_CUDA, "no CUDA device (there is no CPU fallback)")
    f32, i32 = torch.float32, torch.int32
    keep = dict(vert_pos=_dev(inp["vert_pos"], f32), faces=_dev(inp["faces"], i32), vert_normal=_dev(inp.get("vert_normal"), f32),
                vert_skin_w=_dev(inp["vert_skin_w"], f32), vert_disp=_dev(inp.get("vert_disp"), f32),
                vert_albedo=_dev(inp["vert_albedo"], f32), vert_rough=_dev(inp["vert_rough"], f32),
                vert_spec=_dev(inp["vert_spec"], f32), gauss_pos=_dev(inp["gauss_pos"], f32),
                gauss_quat=_dev(inp.get("gauss_quat"), f32), gauss_scale=_dev(inp.get("gauss_scale"), f32),
                gauss_opacity=_dev(inp.get("gauss_opacity"), f32), vert_quat=_dev(inp.get("vert_quat"), f32),
                vert_scale=_dev(inp.get("vert_scale"), f32))
    d = _Desc()
    d.n_verts, d.n_faces = keep["vert_pos"].shape[0], keep["faces"].shape[0]
    d.n_bones, d.n_gauss = keep["vert_skin_w"].shape[1], keep["gauss_pos"].shape[0]
    d.k_g, d.k_v = k_g, k_v
    for k, t in keep.items():
        setattr(d, k, 0 if t is None else t.data_ptr())
    d.max_width, d.max_height, d.max_vis_dirs, d.max_vis_res = max_width, max_height, max_vis_dirs, max_vis_res
    d.max_env_texels, d.max_duplicates = max_env_texels, max_duplicates
    h = C.c_void_p()
    _chk(lib().avatar_load(C.byref(d), _stream(), C.byref(h)))
    del keep                                  # the library copied what it needs
    return h


def avatar_free(h):
    _chk(lib().avatar_free(h))


def pose_skin(h, bone_mats):
    _chk(lib().pose_skin(h, _ptr(bone_mats), _stream()))


def visibility_raster(h, dirs, res, mode=0, depth_bias_texels=1.0, depth_bias_world=0.015, slope_max=8.0, keep_maps=False,
                      cull_backfaces=False):
    p = _VisParams(int(dirs.shape[0]), int(res), int(mode), dirs.data_ptr(), depth_bias_texels, depth_bias_world, slope_max,
                   int(keep_maps), int(cull_backfaces))
    _chk(lib().visibility_raster(h, C.byref(p), _stream()))


def shade_gaussians(h, radiance, cam_pos, texel_to_dir=None, gamma=2.2, use_visibility=True):
    e = _Env(int(radiance.shape[0]), int(radiance.shape[1]), radiance.data_ptr(),
             0 if texel_to_dir is None else texel_to_dir.data_ptr(), gamma, int(use_visibility))
    cp = (C.c_float * 3)(*[float(v) for v in cam_pos])
    _chk(lib().shade_gaussians(h, C.byref(e), cp, _stream()))


def shade_backward(h, radiance, cam_pos, dL_dcolor, texel_to_dir=None, gamma=2.2, use_visibility=True, out_dalbedo=None, out_drough=None,
                   out_dspec=None, out_dnormal=None, out_dpos=None, out_denv=None):
    """Backward of shade_gaussians for the last shaded frame (include/rga.h shade_backward).  All tensors CUDA float32."""
    e = _Env(int(radiance.shape[0]), int(radiance.shape[1]), radiance.data_ptr(),
             0 if texel_to_dir is None else texel_to_dir.data_ptr(), gamma, int(use_visibility))
    cp = (C.c_float * 3)(*[float(v) for v in cam_pos])
    lib().shade_backward.argtypes = [C.c_void_p, C.POINTER(_Env), C.c_float * 3] + [C.c_void_p] * 8
    _chk(lib().shade_backward(h, C.byref(e), cp, _ptr(dL_dcolor), _ptr(out_dalbedo), _ptr(out_drough), _ptr(out_dspec), _ptr(out_dnormal),
                              _ptr(out_dpos), _ptr(out_denv), _stream()))


def splat_render(h, camera, bg, out_image):
    cam = camera if isinstance(camera, _Camera) else make_camera(camera)
    b = (C.c_float * 3)(*[float(v) for v in bg])
    _chk(lib().splat_render(h, C.byref(cam), b, _ptr(out_image), _stream()))


def gaussians_update(h, gauss_pos):
    """Per-frame KNN + Eq.1 re-interpolation for moved Gaussians (include/rga.h gaussians_update)."""
    lib().gaussians_update.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    _chk(lib().gaussians_update(h, _ptr(gauss_pos), _stream()))


def splat_backward(h, camera, bg, image, dL_dimage, out_dcolor=None, out_dopacity=None, out_dmean=None, out_dcov=None):
    """Backward of splat_render for the last rendered frame (include/rga.h splat_backward); image = the tensor that frame was
    rendered into.  All tensors CUDA float32."""
    cam = camera if isinstance(camera, _Camera) else make_camera(camera)
    b = (C.c_float * 3)(*[float(v) for v in bg])
    lib().splat_backward.argtypes = [C.c_void_p, C.POINTER(_Camera), C.c_float * 3] + [C.c_void_p] * 7
    _chk(lib().splat_backward(h, C.byref(cam), b, _ptr(image), _ptr(dL_dimage), _ptr(out_dcolor), _ptr(out_dopacity), _ptr(out_dmean), _ptr(out_dcov),
                              _stream()))


def image_loss(h, image, target, lam=0.2, out_loss=None, out_dL_dimage=None):
    """Eq.5 image loss and its gradient (include/rga.h image_loss).  image, target: CUDA float32 [H, W, 3]."""
    lib().image_loss.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    _chk(lib().image_loss(h, _ptr(image), _ptr(target), int(image.shape[1]), int(image.shape[0]), float(lam), _ptr(out_loss),
                          _ptr(out_dL_dimage), _stream()))


IMAGE_LOSS_STATIC_MAX_PIXELS = 262144


def rga_image_loss_static(image, target, lam=0.2, out_loss=None, out_dL_dimage=None):
    """Eq.5 image loss and its gradient with the library's fixed scratch array: no avatar handle, no allocation
    (include/rga.h rga_image_loss_static; width * height <= IMAGE_LOSS_STATIC_MAX_PIXELS).  image, target: CUDA float32 [H, W, 3]."""
    lib().rga_image_loss_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    _chk(lib().rga_image_loss_static(_ptr(image), _ptr(target), int(image.shape[1]), int(image.shape[0]), float(lam), _ptr(out_loss),
                                     _ptr(out_dL_dimage), _stream()))


def regularisers(h, s0=0.005, out_losses=None, out_dalbedo=None, out_drough=None, out_dspec=None, out_dgauss_pos=None, out_ddisp=None,
                 out_dscale=None):
    """Eq.6-9 and their gradients on the avatar's own tables (include/rga.h regularisers)."""
    lib().regularisers.argtypes = [C.c_void_p, C.c_float] + [C.c_void_p] * 8
    _chk(lib().regularisers(h, float(s0), _ptr(out_losses), _ptr(out_dalbedo), _ptr(out_drough), _ptr(out_dspec), _ptr(out_dgauss_pos),
                            _ptr(out_ddisp), _ptr(out_dscale), _stream()))


class _PosedGrads(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("d_mean", "d_mean2", "d_normal", "d_cov", "d_albedo", "d_rough", "d_spec")]


class _CanonicalGrads(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("d_gauss_pos", "d_gauss_quat", "d_gauss_scale", "d_bones", "d_vert_disp", "d_vert_normal",
                                          "d_vert_albedo", "d_vert_rough", "d_vert_spec")]


def pose_backward(h, bone_mats, posed, canonical):
    """Backward of H2 + Eq.1 (include/rga.h pose_backward).  posed / canonical: dicts of CUDA float32 tensors keyed by the
    field names of rga_posed_grads / rga_canonical_grads; missing keys are NULL."""
    pin = _PosedGrads(*[None if posed.get(n) is None else posed[n].data_ptr() for n, _ in _PosedGrads._fields_])
    pout = _CanonicalGrads(*[None if canonical.get(n) is None else canonical[n].data_ptr() for n, _ in _CanonicalGrads._fields_])
    lib().pose_backward.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_PosedGrads), C.POINTER(_CanonicalGrads), C.c_void_p]
    _chk(lib().pose_backward(h, _ptr(bone_mats), C.byref(pin), C.byref(pout), _stream()))


def densify_density(h, d0, p0, rnd, out_pos, out_tri=None, out_count=None):
    """Algorithm 1, density-based densification (include/rga.h densify_density).  rnd: CUDA int32/uint32 tensor [3 * max_out]
    of raw 32-bit random numbers; out_pos: CUDA float32 [max_out, 3]; out_tri / out_count: CUDA int32 [max_out] / [1] or None."""
    max_out = int(out_pos.shape[0]) if out_pos is not None else 0
    if max_out and rnd.numel() < 3 * max_out:
        raise ValueError("densify_density: rnd needs 3 numbers per output row")
    lib().densify_density.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.c_void_p]
    _chk(lib().densify_density(h, float(d0), float(p0), _ptr(rnd), max_out, _ptr(out_pos), _ptr(out_tri), _ptr(out_count), _stream()))


class _DispMlp(C.Structure):
    _fields_ = [("n_freq", C.c_int32), ("n_pose", C.c_int32), ("rff", C.c_void_p), ("W1", C.c_void_p), ("b1", C.c_void_p),
                ("Wh", C.c_void_p), ("bh", C.c_void_p), ("Wo", C.c_void_p), ("bo", C.c_void_p)]


def displacement_mlp(h, mlp, theta):
    """d(x, theta) on the tensor cores (include/rga.h displacement_mlp).  mlp: dict of CUDA tensors rff, W1, b1, Wh, bh, Wo,
    bo plus n_freq, n_pose; theta: CUDA tensor [n_pose]."""
    m = _DispMlp(int(mlp["n_freq"]), int(mlp["n_pose"]), *[mlp[k].data_ptr() for k in ("rff", "W1", "b1", "Wh", "bh", "Wo", "bo")])
    lib().displacement_mlp.argtypes = [C.c_void_p, C.POINTER(_DispMlp), C.c_void_p, C.c_void_p]
    _chk(lib().displacement_mlp(h, C.byref(m), _ptr(theta), _stream()))


def displacement_static(h):
    """Back to avatar_load's static displacement (include/rga.h displacement_static)."""
    lib().displacement_static.argtypes = [C.c_void_p, C.c_void_p]
    _chk(lib().displacement_static(h, _stream()))


RGA_ATTR_ALBEDO, RGA_ATTR_NORMAL = 1, 2


def splat_attribute(h, camera, bg, which, out_image):
    """Albedo / normal map of the current pose (include/rga.h splat_attribute)."""
    cam = camera if isinstance(camera, _Camera) else make_camera(camera)
    b = (C.c_float * 3)(*[float(v) for v in bg])
    _chk(lib().splat_attribute(h, C.byref(cam), b, int(which), _ptr(out_image), _stream()))


def rga_render_frame(h, bone_mats, dirs, vis_res, radiance, texel_to_dir, cam_pos, camera, bg, out_image, vis_mode=0,
                     use_visibility=True, gamma=2.2, bias=(1.0, 0.015, 8.0), keep_maps=False, cull_backfaces=False):
    """One whole frame in one C-ABI call (include/rga.h rga_render_frame)."""
    e = _Env(int(radiance.shape[0]), int(radiance.shape[1]), radiance.data_ptr(),
             0 if texel_to_dir is None else texel_to_dir.data_ptr(), gamma, int(use_visibility))
    cp = (C.c_float * 3)(*[float(v) for v in cam_pos])
    cam = camera if isinstance(camera, _Camera) else make_camera(camera)
    b = (C.c_float * 3)(*[float(v) for v in bg])
    vp = None
    if use_visibility:
        vp = C.byref(_VisParams(int(dirs.shape[0]), int(vis_res), int(vis_mode), dirs.data_ptr(), bias[0], bias[1], bias[2],
                                int(keep_maps), int(cull_backfaces)))
    _chk(lib().rga_render_frame(h, _ptr(bone_mats), vp, C.byref(e), cp, C.byref(cam), b, _ptr(out_image), _stream()))


def rga_check(h):
    _chk(lib().rga_check(h, _stream()))


def rga_profile_enable(h, on):
    _chk(lib().rga_profile_enable(h, int(on)))


def rga_profile_read(h, capacity=96):
    """-> list of (kernel name, milliseconds) recorded since the last read."""
    names = C.create_string_buffer(32 * capacity)
    ms = (C.c_float * capacity)()
    n = C.c_int(0)
    _chk(lib().rga_profile_read(h, _stream(), names, ms, capacity, C.byref(n)))
    return [(names.raw[32 * i:32 * i + 32].split(b"\0")[0].decode(), float(ms[i])) for i in range(n.value)]


def rga_measure_fp32_peak():
    """Measured FP32 FMA throughput of the current device in TFLOP/s (include/rga.h)."""
    v = C.c_float(0)
    lib().rga_measure_fp32_peak.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    _chk(lib().rga_measure_fp32_peak(_stream(), C.byref(v)))
    return float(v.value)


def rga_launch_count(h):
    return int(lib().rga_launch_count(h))


def rga_read_buffer(h, which):
    """Intermediate buffer -> flat numpy array (host).  Parity tests reshape it as include/rga.h documents."""
    which = BUF[which] if isinstance(which, str) else which
    n = C.c_size_t(0)
    p = C.c_void_p()
    _chk(lib().rga_get_buffer(h, which, _stream(), C.byref(p), C.byref(n)))
    dt = np.dtype(_BUF_DTYPE[which])
    out = np.empty(n.value // dt.itemsize, dt)
    if n.value:
        _chk(lib().rga_read_buffer(h, which, _stream(), out.ctypes.data_as(C.c_void_p), C.c_size_t(out.nbytes), C.byref(n)))
    return out


class Avatar:
    """Convenience owner of an rga_avatar handle plus the device copies of per-frame inputs."""

    def __init__(self, inp, **maxima):
        self.h = avatar_load(inp, **maxima)

    def close(self):
        if self.h is not None:
            avatar_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def render(self, bone_mats, dirs, vis_res, radiance, texel_to_dir, cam_pos, camera, bg, out_image, vis_mode=0,
               use_visibility=True, gamma=2.2, bias=(1.0, 0.015, 8.0), cull_backfaces=False):
        """One relit posed frame through rga_render_frame."""
        rga_render_frame(self.h, bone_mats, dirs, vis_res, radiance, texel_to_dir, cam_pos, camera, bg, out_image, vis_mode,
                         use_visibility, gamma, bias, cull_backfaces=cull_backfaces)
        return out_image

    def read(self, which):
        return rga_read_buffer(self.h, which)
