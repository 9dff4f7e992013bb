"""Randomised parity sweep on the GPU: `synth.workloads.make_random` draws everything the hot path is parameterised by
(direction grids that are not multiples of 32, odd depth-map sides, images that are not multiples of the tile, close-up and
oblique cameras, off-centre principal points, large Gaussians, bias constants, missing vertex normals) and every stage of
both call styles -- the four stage calls and rga_render_frame -- is compared with the oracle as in test_gpu_parity.py:
integers bit for bit, image / radiance within the north_star tolerances.  A 400-seed run of the same sweep during
development found no mismatch; the 24 seeds kept here take about half a minute."""
import numpy as np
import pytest

from synth import workloads

pytestmark = pytest.mark.gpu

# flagged pixels (A38) per blended (pixel, entry) pair: the 400-seed sweep saw 2e-6 .. 6e-6 where any were flagged
FLAG_PER_PAIR = 2e-5


# seed 9489 (found by a 11,600-seed run): a light almost exactly opposite the viewer, |w_i + w_o| = 0.004 -- the stand-alone shading
# kernel formed |w_i + w_o|^2 as 2 + 2 w_o.w_i there and lost the half vector to cancellation (6e-3 in the radiance)
# seeds 54952 and 56494 (an 18,256-seed run on the round's final build, no wrong output): ONE light direction that stands behind
# every camera-facing Gaussian (nothing for the fused kernel to test: all its words must be 0), and a frame with 3 flagged pixels
# seed 109469 (24,646 more seeds): a pixel whose STOPPING decision can flip (flag bit 1) and does: 7.7e-3, inside what that decision moves
@pytest.mark.parametrize("seed", list(range(24)) + [9489, 54952, 56494, 109469])
def test_random_configuration(seed):
    import torch
    from oracle import oracle as orc
    from paper_2407_10707_b200 import binding as rga
    from parity_util import compare_all, run_gpu
    inp, desc = workloads.make_random(seed)
    mode = 1 if seed % 3 == 2 else 0
    orc_av = orc.avatar_load(inp)
    o = orc.render_frame(orc_av, inp, vis_mode=mode)
    av, img = run_gpu(inp, vis_mode=mode)
    print(desc, compare_all(inp, av, img, orc_av, o, mode, flag_per_pair=FLAG_PER_PAIR))
    av.close()
    if mode != 0:
        return
    cam = inp["camera"]; W, H = cam["width"], cam["height"]
    av = rga.Avatar(inp, max_width=W, max_height=H, max_vis_dirs=len(inp["vis_dirs"]), max_vis_res=inp["vis_res"],
                    max_env_texels=inp["env_rows"] * inp["env_cols"])
    im = torch.empty((H, W, 3), dtype=torch.float32, device="cuda")
    av.render(torch.as_tensor(inp["bone_mats"][0]).cuda(), torch.as_tensor(inp["vis_dirs"]).cuda(), inp["vis_res"],
              torch.as_tensor(inp["env"][0]).cuda(), torch.as_tensor(inp["texel_to_dir"]).cuda(), inp["cam_pos"], cam, inp["bg"], im,
              vis_mode=0, gamma=inp["gamma"], bias=(inp["depth_bias_texels"], inp["depth_bias_world"], inp["slope_max"]))
    rga.rga_check(av.h)
    kept = ((inp["cam_pos"][None, :].astype(np.float64) - o["gauss_posed"]) * o["gauss_normal_posed"]).sum(1) > 0
    if kept.sum() > 32:                                    # a camera that sees no front face leaves nothing to compare bit by bit
        compare_all(inp, av, im.cpu().numpy(), orc_av, o, 0, frame_call=True, flag_per_pair=FLAG_PER_PAIR)
    av.close()
