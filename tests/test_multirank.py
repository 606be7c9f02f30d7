"""N > 1 host logic on CPU (gloo, world_size 2): the path does not exchange data between GPUs
 -- ranks stream independent seeded skies and bench.py only aggregates the
timing (max over ranks), the launch count (sum) and the whole-job frames/s."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _torchrun(args, timeout, attempts=3):
    """torchrun on a fresh port; the port found free can be taken again before the rendezvous binds it, so a failed
    rendezvous (not a failed worker) is tried again on another port."""
    r = None
    for _ in range(attempts):
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
               "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
        r = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=dict(os.environ, OMP_NUM_THREADS="1"), cwd=ROOT)
        if r.returncode == 0 or not any(k in r.stderr for k in ("address already in use", "EADDRINUSE", "Connection refused", "RendezvousConnectionError", "failed to bind", "DistNetworkError")):
            break
    return r


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, world, _ = bench.env_rank()
dist.init_process_group("gloo", rank=rank, world_size=world)
# rank r pretends its K steps took 10 + 5 r ms and launched 12 (r + 1) kernels
ms, launches = bench.reduce_over_ranks(10.0 + 5.0 * rank, 12 * (rank + 1), "cpu", world)
from paper_2103_15418_b200 import synth
s = synth.CubeStream(1, seed=bench.rank_seed(rank))
cube = s.frame(0)
out = dict(rank=rank, ms=ms, launches=launches, value=bench.whole_job_value(world, 100, ms),
           checksum=float(cube.astype("float64").sum()))
dist.barrier()
# one file per rank: two ranks printing to the same pipe can interleave inside a line
open(os.path.join({out!r}, "rank%d.json" % rank), "w").write(json.dumps(out))
dist.destroy_process_group()
"""


def test_two_ranks_gloo_aggregation(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, out=str(tmp_path)))
    r = _torchrun([str(script)], timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.loads((tmp_path / f"rank{k}.json").read_text()) for k in range(2)]
    assert sorted(x["rank"] for x in res) == [0, 1]
    for x in res:
        assert x["ms"] == 15.0            # max over ranks
        assert x["launches"] == 36        # sum over ranks
        assert abs(x["value"] - 2 * 100 / 0.015) < 1e-6   # whole-job frames/s
    # weak scaling: every rank streams its own seeded sky
    assert res[0]["checksum"] != res[1]["checksum"]


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """`bench.py --impl reference` under torchrun: rank 0 alone runs the oracle and prints ONE JSON line."""
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "3", "--config", "1"],
                  timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "frames/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_single_rank_helpers():
    import bench
    assert bench.reduce_over_ranks(3.5, 7, "cpu", 1) == (3.5, 7)
    assert bench.whole_job_value(4, 10, 20.0) == 4 * 10 / 0.02
    assert [bench.rank_seed(r) for r in range(3)] == [0, 1, 2]
