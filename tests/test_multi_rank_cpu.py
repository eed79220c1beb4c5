"""N > 1 host logic on CPU (gloo, world_size 2): rank setup from the torchrun environment, one seeded population per
rank (weak scaling, no data-path collective), barrier + max-over-ranks timing, whole-job aggregation, and the
reference arm running on rank 0 only.  No CUDA call is made here."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["PT_ROOT"])
import numpy as np
import torch
import bench
from paper_1504_07433_b200 import inputs

rank, world, local = bench._dist_setup(2)
dev = torch.device("cpu")
w = inputs.config2(n_pv=4, n_t=100, stream=rank)          # the bench's per-rank population
fake_seconds = 1.0 + rank                                   # rank 1 is the slow one
bench._barrier(world)                                       # must not need CUDA on a CPU box
t_max = bench._max_over_ranks(fake_seconds, world, dev)
value = world * w.n_eval * 3 / t_max                        # bench.py's whole-job aggregate for 3 steps
import torch.distributed as dist
digest = torch.tensor([float(np.sum(w.params))], dtype=torch.float64)
both = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
dist.all_gather(both, digest)
print(json.dumps({"rank": rank, "world": world, "local": local, "t_max": t_max, "value": value,
                  "digests": [float(b) for b in both]}), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _spawn(code_or_args, world=2, is_code=True):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), PT_ROOT=ROOT, CUDA_VISIBLE_DEVICES="")
        cmd = [sys.executable, "-c", code_or_args] if is_code else [sys.executable] + code_or_args
        procs.append(subprocess.Popen(cmd, env=env, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_two_ranks_gloo_timing_and_sharding():
    outs = _spawn(WORKER)
    res = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    assert [d["rank"] for d in res] == [0, 1] and all(d["world"] == 2 for d in res)
    # max over ranks: both ranks agree on the slow rank's time
    assert all(d["t_max"] == 2.0 for d in res)
    # whole-job value = units of all ranks / max time
    assert all(d["value"] == 2 * (4 * 100 * 10) * 3 / 2.0 for d in res)
    # every rank evaluated its own population (different seeds), and both saw the same pair
    assert res[0]["digests"] == res[1]["digests"] and res[0]["digests"][0] != res[0]["digests"][1]


def test_reference_arm_runs_on_rank0_only():
    outs = _spawn(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"], is_code=False)
    lines = [o.strip() for o in outs]
    assert lines[1] == ""                                    # rank 1 exits 0 without work
    d = json.loads(lines[0].splitlines()[-1])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_per_rank_populations_are_disjoint_streams():
    from paper_1504_07433_b200 import inputs
    a, b = inputs.config2(stream=0), inputs.config2(stream=1)
    assert a.params.shape == b.params.shape and not np.array_equal(a.params, b.params)
    assert a.n_eval == b.n_eval == 38400000
