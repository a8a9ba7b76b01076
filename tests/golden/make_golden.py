#!/usr/bin/env python
"""Writes tests/golden/cfg1_oracle.txt: a digest of the CPU oracle's outputs on BASELINE.json configs[0]
(the tiny scene) and on the smoke scene.  Calls ONLY oracle/ and the seeded generator workloads/ -- never the CUDA path.

    python tests/golden/make_golden.py

The paper (arxiv/paper_2606_15924) prints no worked numeric example of the rasterisation (its tables are
dataset metrics), so no value here is the paper's; the file pins the oracle against silent change: any edit of
its arithmetic moves these numbers and has to be justified in the commit that regenerates them
(tests/test_oracle_pins.py::test_golden_digest_of_the_tiny_scene compares).
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads  # noqa: E402


SCENES = {
    "cfg1": lambda: workloads.make(1),  # BASELINE.json configs[0]; its top-error tiles are the nearly empty ones
    "small_rot": lambda: workloads.small_random_scene(7, 3000, 200, 136, sh_degree=3, bg=(0.1, 0.3, 0.2), spread=1.3,
                                                       log_scale=(-2.8, 0.6)),  # the smoke scene: a real multi-layer composite
}


def digest(name):
    o = oracle.Oracle("f32")
    sc = SCENES[name]()
    r = o.pipeline(sc, backward=False, restrict=True)
    g = workloads.dl_dcolor(0, r.samp.n)
    name_ = name + "."
    rb = o.raster_bwd(sc.cam, r.binned, r.pre, r.samp, r.fwd, g)
    pb = o.project_bwd(sc.cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.sh, r.pre.radii, r.pre.clamped,
                       rb.dL_dmeans2D, rb.dL_dconic, rb.dL_drgb)
    sha = lambda a: hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:16]
    lines = [
        ("P", int(r.binned.P)), ("k", int(r.samp.k)), ("n", int(r.samp.n)),
        ("sha_rect", sha(r.pre.rect)), ("sha_depth_bits", sha(r.pre.depths.astype(np.float32).view(np.uint32))),
        ("sha_tile_offsets", sha(r.binned.tile_offsets)), ("sha_gid_sorted", sha(r.binned.gid_sorted)),
        ("sha_tiles", sha(r.samp.tiles)), ("sha_pix", sha(r.samp.pix)),
        ("sum_color", f"{float(r.fwd.color.astype(np.float64).sum()):.6f}"),
        ("sum_T", f"{float(r.fwd.T.astype(np.float64).sum()):.6f}"),
        ("sum_n_contrib", int(r.fwd.n_contrib.astype(np.int64).sum())),
        ("l1_dL_dmeans3D", f"{float(np.abs(pb.dL_dmeans3D.astype(np.float64)).sum()):.6e}"),
        ("l1_dL_dscales", f"{float(np.abs(pb.dL_dscales.astype(np.float64)).sum()):.6e}"),
        ("l1_dL_dquats", f"{float(np.abs(pb.dL_dquats.astype(np.float64)).sum()):.6e}"),
        ("l1_dL_dsh", f"{float(np.abs(pb.dL_dsh.astype(np.float64)).sum()):.6e}"),
    ]
    return [(name_ + k, v) for k, v in lines]


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle.txt")
    with open(out, "w") as f:
        f.write("# digest of the CPU oracle (fp32 build) on BASELINE.json configs[0]; written by tests/golden/make_golden.py\n")
        f.write("# (oracle/ only; no value from the CUDA path, none from the paper: it prints no worked example)\n")
        for name in SCENES:
            for k, v in digest(name):
                f.write(f"{k} {v}\n")
    print(open(out).read())
