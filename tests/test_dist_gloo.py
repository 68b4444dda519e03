"""N > 1 plumbing on CPU: two gloo processes (the bench's barrier, max-over-ranks timing and
row ownership), and `bench.py --impl reference` under a 2-rank launch (rank 0 alone works).

The path has no data-path collective: the only things that cross
ranks are a barrier and the max of a scalar time, which is what these tests cover.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np
from paper_2607_02521_b200 import dist, inputs
r = dist.Ranks(backend="gloo")
r.barrier()
slow = r.max_over_ranks(10.0 + 5.0 * r.rank)        # rank 1 is the slow one
total = r.sum_over_ranks(float(r.rank + 1))
# weak scaling row ownership used by bench.Workload: rank r owns rows [r*M, (r+1)*M)
M, K, seed = 5, 64, 3
mine = inputs.make_activations((r.rank + 1) * M, K, seed)[r.rank * M:]
r.barrier()
print(json.dumps({{"rank": r.rank, "world": r.world, "slow": slow, "total": total,
                  "rows_crc": int(mine.astype(np.uint64).sum())}}))
r.close()
"""


def _launch(script: str, world: int = 2, timeout: int = 120):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, WORLD_SIZE=str(world), RANK=str(rank), LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", script], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=timeout)
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    return outs


def test_two_gloo_ranks_barrier_max_time_and_row_ownership():
    from paper_2607_02521_b200 import inputs
    outs = _launch(_WORKER.format(root=ROOT))
    recs = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    assert [d["rank"] for d in recs] == [0, 1] and all(d["world"] == 2 for d in recs)
    assert all(d["slow"] == 15.0 for d in recs)      # every rank sees the slowest rank's time
    assert all(d["total"] == 3.0 for d in recs)
    # the two ranks own DIFFERENT rows of the same seeded stream
    allA = inputs.make_activations(10, 64, 3)
    assert recs[0]["rows_crc"] == int(allA[:5].astype(np.uint64).sum())
    assert recs[1]["rows_crc"] == int(allA[5:].astype(np.uint64).sum())
    assert recs[0]["rows_crc"] != recs[1]["rows_crc"]


def test_reference_arm_under_two_ranks_only_rank0_prints():
    """`bench.py --impl reference` launched as 2 ranks: rank 0 times the oracle and prints the
    JSON line, rank 1 exits 0 without work (tier contract)."""
    port = _free_port()
    outs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="",
                   SWIGLU_REFERENCE_BUDGET_S="2")
        p = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "0", "--workload", "qwen2.5-0.5b"],
                           env=env, cwd=ROOT, capture_output=True, text=True, timeout=300)
        assert p.returncode == 0, p.stderr[-2000:]
        outs.append(p.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
