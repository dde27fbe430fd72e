"""Multi-GPU is "replicas only": one independent magnetogram per rank, no data-path
collective; bench.py only reduces the time (MAX) and the cycle count (SUM) over ranks.  This covers that
host-side logic with a world_size-2 gloo run on CPU: distinct seeded inputs per rank, the reductions, and
that rank 0 alone reports."""
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import json, os, sys
sys.path.insert(0, os.environ["MHS_ROOT"])
import numpy as np
import torch
import torch.distributed as dist
import bench
from paper_1307_6720_b200 import inputs
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = inputs.config(1, shrink=8, replica=rank)
ms, cycles = bench.reduce_over_ranks(10.0 + 5.0 * rank, 7 + rank, world, device="cpu")
digest = float(np.abs(w.Bz0).sum())
all_d = [None] * world
dist.all_gather_object(all_d, digest)
if rank == 0:
    print(json.dumps({"ms": ms, "cycles": cycles, "digests": all_d, "mean": float(w.Bz0.mean())}))
dist.destroy_process_group()
'''


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_replica_reduction_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MHS_ROOT=ROOT, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout          # rank 0 alone prints
    import json
    r = json.loads(lines[0])
    assert r["ms"] == 15.0                      # MAX over ranks
    assert r["cycles"] == 15                    # SUM over ranks (7 + 8)
    assert abs(r["digests"][0] - r["digests"][1]) > 1e-6   # independent magnetograms
    assert abs(r["mean"]) < 1e-12               # net flux zeroed (C18)


def test_replica_zero_is_the_config_itself():
    from paper_1307_6720_b200 import inputs
    a, b = inputs.config(1, shrink=8), inputs.config(1, shrink=8, replica=0)
    assert np.array_equal(a.Bz0, b.Bz0)
    c = inputs.config(1, shrink=8, replica=1)
    assert not np.array_equal(a.Bz0, c.Bz0) and np.array_equal(a.f, c.f)
