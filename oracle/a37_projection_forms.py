"""Reading A37: how much do the oracle's two restatements of the light-space projection and of the depth-test
bias move?  Round 1 rewrote `light_project` / beta from the spelled-out form of SURVEY.md:371-381
    px = ((u.d)/r * 1/2 + 1/2) R_v,   z = (r - w.d)/(2r),   beta = ((bias_texels (2r/R_v)) tau + bias_world)/(2r)
to three fused multiply-add chains on a per-direction pre-scaled frame (oracle/rga_oracle.cpp `light_project`).  Both are
the same real-valued function; they differ only in fp32 rounding.  This script runs the ORACLE ALONE on configs 0 and 1
in both forms and counts the depth-map texels, triangle ids and visibility bits that differ.

    python -m oracle.a37_projection_forms            # prints one line per config; `--write` refreshes tests/golden/a37_projection_forms.txt

Calls only oracle/ and synth/ (inputs).  TEST INFRASTRUCTURE."""
import os
import sys

import numpy as np

from oracle import oracle as orc
from synth import workloads


def count(cfg, n_gauss=None):
    inp = workloads.make(cfg, n_gauss=n_gauss)
    av = orc.avatar_load(inp)
    out = []
    for plain in (0, 1):
        orc.lib().orc_set_plain_projection(plain)
        try:
            out.append(orc.render_frame(av, inp, vis_mode=0, stop_after="vis"))
        finally:
            orc.lib().orc_set_plain_projection(0)
    a, b = out
    cov_a, cov_b = a["zmap"] != 0xFFFFFFFF, b["zmap"] != 0xFFFFFFFF
    both = cov_a & cov_b
    za, zb = a["zmap"].view(np.float32), b["zmap"].view(np.float32)
    K = len(inp["vis_dirs"])
    xa = ((a["visbits"][:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(len(a["visbits"]), -1)[:, :K]
    xb = ((b["visbits"][:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(len(b["visbits"]), -1)[:, :K]
    return dict(cfg=cfg, texels=int(cov_a.size), covered=int(cov_a.sum()), coverage_differs=int((cov_a != cov_b).sum()),
                depth_bits_differ=int((a["zmap"] != b["zmap"]).sum()), id_differs=int((a["idmap"] != b["idmap"]).sum()),
                max_abs_depth_diff=float(np.abs(za[both].astype(np.float64) - zb[both]).max()),
                vis_bits=int(xa.size), vis_bits_differ=int((xa != xb).sum()))


def main():
    rows = [count(0), count(1)]
    for r in rows:
        print(r)
    if "--write" in sys.argv:
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "tests", "golden", "a37_projection_forms.txt")
        with open(path, "w") as f:
            f.write("# written by `python -m oracle.a37_projection_forms --write` (oracle only; DESIGN.md reading A37)\n")
            f.write("# fused form (current oracle) vs the spelled-out form of SURVEY.md:371-381\n")
            f.write("# cfg texels covered coverage_differs depth_bits_differ id_differs max_abs_depth_diff vis_bits vis_bits_differ\n")
            for r in rows:
                f.write("%d %d %d %d %d %d %.3e %d %d\n" % (r["cfg"], r["texels"], r["covered"], r["coverage_differs"], r["depth_bits_differ"],
                                                          r["id_differs"], r["max_abs_depth_diff"], r["vis_bits"], r["vis_bits_differ"]))


if __name__ == "__main__":
    main()
