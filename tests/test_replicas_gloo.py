"""N > 1 path of bench.py ("replicas only") on CPU: two gloo ranks run the measurement
plumbing of paper_2510_02483_b200.replicas -- rendezvous on 127.0.0.1, barrier, MAX over ranks of the per-rank
time, SUM over ranks of the units -- and the reference arm's "rank 0 alone prints" rule."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["LSP_ROOT"])
from paper_2510_02483_b200 import replicas
renv = replicas.rank_env()
assert replicas.init("gloo", renv)
replicas.barrier()
ms_local = 10.0 + 5.0 * renv.rank                 # rank 1 is the slow one
value, ms_max, units = replicas.whole_job_throughput(1000.0, ms_local)
replicas.barrier()
print(json.dumps(dict(rank=renv.rank, main=renv.is_main, value=value, ms_max=ms_max, units=units)), flush=True)
replicas.finalize()
"""


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_rank_env_defaults():
    from paper_2510_02483_b200 import replicas
    e = replicas.rank_env({})
    assert (e.rank, e.local_rank, e.world_size, e.is_main) == (0, 0, 1, True)
    e = replicas.rank_env({"RANK": "3", "LOCAL_RANK": "1", "WORLD_SIZE": "4"})
    assert (e.rank, e.local_rank, e.world_size, e.is_main) == (3, 1, 4, False)
    # single process: no group, the reductions are the identity
    assert replicas.whole_job_throughput(500.0, 250.0) == (2000.0, 250.0, 500.0)


@pytest.mark.timeout(180)
def test_two_gloo_ranks_max_time_sum_units():
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), LSP_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=150)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms_max"] == 15.0                 # MAX over ranks, not this rank's own time
        assert o["units"] == 2000.0                # all ranks' units
        assert abs(o["value"] - 2000.0 / 15e-3) < 1e-6
    assert sorted(o["main"] for o in outs) == [False, True]


@pytest.mark.timeout(180)
def test_reference_arm_rank1_prints_nothing():
    """bench.py --impl reference under torchrun: ranks other than 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=150)
    assert r.returncode == 0, r.stderr
    assert r.stdout.strip() == ""
