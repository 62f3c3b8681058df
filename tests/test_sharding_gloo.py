"""N > 1 path on CPU: two processes over gloo run the benchmark's multi-rank plumbing (paper_2606_29207_b200.sharding):
per-rank independent batches, time = MAX over ranks, bytes / launches = SUM over ranks.  The path itself has no
data-path collective, so this is all the distributed logic there is."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, os.environ["KF_ROOT"])
    import torch.distributed as dist
    from kf_inputs import gen, workloads
    from paper_2606_29207_b200 import sharding
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = workloads.by_name("cfg3")
    wl.seed = sharding.rank_seed(wl.seed, rank)
    q = gen.gen_q(0, 0, 0, wl.n_q_heads, wl.seed)                 # this rank's inputs
    ms_local, bytes_local, launches_local = 10.0 + 5.0 * rank, 1e9 * (rank + 1), 100 + rank
    dist.barrier()
    ms, nbytes, launches = sharding.aggregate(ms_local, bytes_local, launches_local, dist)
    out = {"rank": rank, "ms": ms, "bytes": nbytes, "launches": launches, "gbs": sharding.throughput_gbs(nbytes, ms),
           "q_sum": float(abs(q.astype("float64")).sum()), "seed": wl.seed, "contexts": wl.contexts[:3]}
    dist.barrier()
    dist.destroy_process_group()
    print("RESULT " + json.dumps(out))
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_aggregation_over_gloo():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   KF_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        res.append(json.loads([l for l in out.splitlines() if l.startswith("RESULT ")][0][7:]))
    res.sort(key=lambda r: r["rank"])
    for r in res:                                   # every rank sees the same whole-job numbers
        assert r["ms"] == 15.0                      # max(10, 15)
        assert r["bytes"] == 3e9                    # 1e9 + 2e9
        assert r["launches"] == 201
        assert np.isclose(r["gbs"], 3e9 / 15e-3 / 1e9)
    # independent batches: different seeds -> different inputs, same recipe shape
    assert res[0]["seed"] + 1 == res[1]["seed"]
    assert res[0]["q_sum"] != res[1]["q_sum"]
    assert res[0]["contexts"] == res[1]["contexts"]     # same length recipe on every rank: balanced weak scaling


def test_single_process_aggregate_is_identity():
    from paper_2606_29207_b200 import sharding
    assert sharding.aggregate(3.5, 7e9, 42, None) == (3.5, 7e9, 42)
    assert sharding.rank_seed(260629207, 0) == 260629207
