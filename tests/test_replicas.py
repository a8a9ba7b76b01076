"""N > 1 is "replicas only": what ranks share is the measurement plumbing.  This
covers it with two gloo processes on CPU: barrier, max-over-ranks time, sum-over-ranks units, one view per rank."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["TGS_ROOT"])
import torch
from paper_2606_15924_b200.replicas import Replicas
rep = Replicas("gloo", torch.device("cpu"))
rep.barrier()
ms = 10.0 + 5.0 * rep.rank            # rank 1 is the slow one
units = 1000.0 * (rep.rank + 1)       # ranks process different amounts
out = {"rank": rep.rank, "world": rep.world, "seed": rep.view_seed(40),
       "max_ms": rep.max_over_ranks(ms), "sum_units": rep.sum_over_ranks(units),
       "value": rep.throughput(units, 4, ms)}
rep.barrier()
rep.close()
print("RESULT " + json.dumps(out))
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_replica_plumbing_world_size_2_gloo(tmp_path):
    import json
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), TGS_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    res = {}
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0, out
        line = [ln for ln in out.splitlines() if ln.startswith("RESULT ")][-1]
        d = json.loads(line[7:])
        res[d["rank"]] = d
    assert set(res) == {0, 1}
    for r, d in res.items():
        assert d["world"] == 2 and d["seed"] == 40 + r          # one view per rank
        assert d["max_ms"] == 15.0                              # the slowest rank's time
        assert d["sum_units"] == 3000.0                         # whole-job units
        assert abs(d["value"] - 3000.0 * 4 / 15e-3) < 1e-6      # whole-job throughput, same on every rank


def test_single_process_is_the_identity():
    import torch
    from paper_2606_15924_b200.replicas import Replicas
    env = {k: os.environ.pop(k, None) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    try:
        rep = Replicas("gloo", torch.device("cpu"))
        assert rep.world == 1 and rep.max_over_ranks(3.5) == 3.5 and rep.sum_over_ranks(7) == 7.0
        assert rep.throughput(100, 2, 50.0) == 100 * 2 / 50e-3
        rep.barrier()
        rep.close()
    finally:
        for k, v in env.items():
            if v is not None:
                os.environ[k] = v


def test_one_view_per_rank_orbits_the_scene():
    """bench.py hands Replicas.view_seed(0) to workloads.orbit_view: rank 0 keeps the config's own camera, rank r > 0
    sees the same Gaussians from another seeded direction at the same distance, through the oracle's projection."""
    import numpy as np
    import oracle
    import workloads
    sc = workloads.make(2)
    assert workloads.orbit_view(sc, 0) is sc
    o = oracle.Oracle("f32")
    seen = []
    for view in (0, 1, 2):
        v = workloads.orbit_view(sc, view)
        R = np.asarray(v.cam.R, np.float64)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-6) and abs(np.linalg.det(R) - 1.0) < 1e-6    # a rotation
        assert np.array_equal(v.cam.t, sc.cam.t) and v.means3D is sc.means3D                      # same distance, same scene
        pre = o.preprocess(v.cam, v.sh_degree, v.means3D, v.scales, v.quats, v.opacities, v.sh)
        vis = pre.radii > 0
        assert vis.mean() > 0.3                                                                   # the cloud stays in view
        seen.append(vis)
    assert (seen[0] != seen[1]).any() and (seen[1] != seen[2]).any()                              # different views
