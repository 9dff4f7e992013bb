"""CPU-side checks: the C-ABI library builds, loads, and exports every symbol include/rga.h declares; the binding's
struct layouts match the header; the product path refuses to run without CUDA (no fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2407_10707_b200 import build
    return build.build()


def test_every_declared_symbol_is_exported(built_lib):
    hdr = open(os.path.join(ROOT, "include", "rga.h")).read()
    names = re.findall(r"RGA_API\s+[\w\s\*]+?\b(\w+)\s*\(", hdr)
    assert {"avatar_load", "pose_skin", "visibility_raster", "shade_gaussians", "splat_render"} <= set(names)
    lib = C.CDLL(built_lib)
    for n in names:
        assert hasattr(lib, n), "librga.so does not export %s" % n
    lib.rga_version.restype = C.c_char_p
    assert b"sm_100a" in lib.rga_version()


def test_binding_struct_layouts_match_header(built_lib):
    from paper_2407_10707_b200 import binding as rga
    assert C.sizeof(rga._Camera) == 9 * 4 + 3 * 4 + 4 * 4 + 2 * 4 + 4
    assert C.sizeof(rga._VisParams) == 48 and rga._VisParams.dirs.offset == 16 and rga._VisParams.cull_backfaces.offset == 40
    assert C.sizeof(rga._Env) == 32 and rga._Env.radiance.offset == 8
    assert rga._Desc.vert_pos.offset == 24 and rga._Desc.max_width.offset == 24 + 12 * 8
    assert C.sizeof(rga._Desc) == 24 + 12 * 8 + 5 * 4 + 4 + 8 + 2 * 8 and rga._Desc.vert_quat.offset == 24 + 12 * 8 + 5 * 4 + 4 + 8
    hdr = open(os.path.join(ROOT, "include", "rga.h")).read()
    ids = dict((m.group(1), int(m.group(2))) for m in re.finditer(r"RGA_BUF_(\w+?)\s*=\s*(\d+)", hdr))
    for k, v in rga.BUF.items():
        assert ids[k] == v


def test_no_cpu_fallback(built_lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_2407_10707_b200 import binding as rga
    from synth import workloads
    with pytest.raises(rga.RgaError):
        rga.avatar_load(workloads.make(0), 64, 64, 16, 64, 128)
    # the raw entry points refuse as well
    lib = C.CDLL(built_lib)
    h = C.c_void_p()
    d = rga._Desc(); d.n_verts = d.n_faces = d.n_bones = d.n_gauss = 1; d.k_g = 3; d.k_v = 19
    for f in ("vert_pos", "faces", "vert_normal", "vert_skin_w", "vert_albedo", "vert_rough", "vert_spec", "gauss_pos",
              "gauss_quat", "gauss_scale"):
        setattr(d, f, 8)
    d.max_width = d.max_height = d.max_vis_dirs = d.max_vis_res = d.max_env_texels = 16
    assert lib.avatar_load(C.byref(d), None, C.byref(h)) == rga.RGA_ERR_CUDA and not h.value


def test_product_package_never_touches_oracle():
    pkg = os.path.join(ROOT, "paper_2407_10707_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src and "rga_oracle" not in src, f


def test_workload_shapes_match_baseline_configs():
    from synth import workloads
    c0 = workloads.make(0)
    assert c0["vert_pos"].shape == (642, 3) and c0["faces"].shape == (1280, 3) and c0["gauss_pos"].shape == (2000, 3)
    assert c0["env"].shape == (1, 8, 16, 3) and c0["vis_dirs"].shape == (16, 3) and c0["vis_res"] == 64
    c1 = workloads.make(1, n_gauss=1000)
    assert c1["vert_pos"].shape == (6890, 3) and c1["faces"].shape == (13776, 3) and c1["n_bones"] == 24
    assert c1["vis_dirs"].shape == (512, 3) and c1["camera"]["width"] == 512
    assert np.allclose(c1["vert_skin_w"].sum(1), 1) and (np.count_nonzero(c1["vert_skin_w"], axis=1) <= 2).all()
    c3 = workloads.make(3, n_gauss=1000)
    assert c3["bone_mats"].shape == (64, 24, 12) and c3["env"].shape[0] == 4 and c3["env_of_frame"].max() <= 3
    assert np.array_equal(c1["texel_to_dir"], np.arange(512))
    # deterministic
    assert np.array_equal(workloads.make(0)["gauss_pos"], c0["gauss_pos"])


def test_argument_checks_need_no_device(built_lib):
    # invalid arguments are rejected before any CUDA call: the status is the same with or without a GPU
    from paper_2407_10707_b200 import binding as rga
    lib = rga.lib()
    assert lib.rga_render_frame(None, None, None, None, None, None, None, None, None) == rga.RGA_ERR_INVALID_ARG
    assert lib.pose_skin(None, None, None) == rga.RGA_ERR_INVALID_ARG
    assert lib.rga_check(None, None) == rga.RGA_ERR_INVALID_ARG
    assert b"null" in lib.rga_last_error()
    h = C.c_void_p()
    d = rga._Desc(); d.n_verts = d.n_faces = d.n_bones = d.n_gauss = 4; d.k_g = 3; d.k_v = 19
    for f in ("vert_pos", "faces", "vert_normal", "vert_skin_w", "vert_albedo", "vert_rough", "vert_spec", "gauss_pos",
              "gauss_quat", "gauss_scale"):
        setattr(d, f, 8)
    d.max_width = d.max_height = d.max_vis_dirs = d.max_env_texels = 16
    d.max_vis_res = 512                                           # snapped raster coordinates are 16-bit: R <= 256
    assert lib.avatar_load(C.byref(d), None, C.byref(h)) == rga.RGA_ERR_INVALID_ARG and not h.value
    d.max_vis_res = 64; d.n_verts = 1 << 21                       # three vertex indices share one 64-bit packed face
    assert lib.avatar_load(C.byref(d), None, C.byref(h)) == rga.RGA_ERR_INVALID_ARG and b"2^21" in lib.rga_last_error()
    # (a mesh whose vertex table exceeds the rasteriser's shared memory is no longer refused: the table then lives in an
    # L2-resident scratch buffer -- tests/test_gpu_parity.py::test_mesh_larger_than_the_shared_memory_vertex_table)
    d.n_verts = 4; d.k_v = 4                                      # the median of Eq.3 needs an odd K_v
    assert lib.avatar_load(C.byref(d), None, C.byref(h)) == rga.RGA_ERR_INVALID_ARG
