"""world_size-2 gloo test of the N>1 host logic of bench.py: chains shard across ranks
with no data-path collective (each rank owns its own chains of the same target), the step time is the
max over ranks, and the reference arm runs on rank 0 only."""
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
spec = dict(bench.WORKLOADS["tiny_mala"])
w, chain0 = bench.shard_workload(spec, rank, world)
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")
dist.barrier()
# the Philox stream this rank's chain 0 draws at step 0 (the stream layout is the oracle's, KAT-pinned)
from oracle import oracle as O
first = O.normals(7, chain0 + 0, 0, w.d)
# the one exchange step of the sharded path (SURVEY 8(e), best_set_adaptation_exchange): every rank's packet of
# window sums, rank order -- here on CPU tensors over gloo, on the GPU box the same call over NCCL
from paper_2606_04895_b200 import distributed as D
send = torch.arange(5, dtype=torch.float64) + 100.0 * rank
recv = torch.zeros(5 * world, dtype=torch.float64)
D.allgather_packets(send, recv)
out = dict(gathered=recv.tolist(), rank=rank, n_chains=int(w.n_chains), theta_sum=float(np.abs(w.theta0).sum()),
           W0=float(w.W[0].sum()), mu0=float(w.mu[0]), ms=ms, chain0=int(chain0), first=[float(x) for x in first])
print("RESULT " + json.dumps(out), flush=True)
dist.destroy_process_group()
"""


def test_sharding_and_max_over_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    import socket
    for attempt in range(3):             # the rendezvous port can be taken between probing and binding: retry
        with socket.socket() as sk:      # a free port: back-to-back runs must not collide
            sk.bind(("127.0.0.1", 0))
            port = str(sk.getsockname()[1])
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=port, OMP_NUM_THREADS="1")
        p = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                            "--master-addr", "127.0.0.1", "--master-port", port, str(script), ROOT],
                           capture_output=True, text=True, timeout=300, env=env)
        if p.returncode == 0:
            break
    assert p.returncode == 0, p.stderr[-2000:]
    import json
    import re                            # the two ranks share stdout: their lines can run into each other
    res = sorted((json.loads(m) for m in re.findall(r"RESULT (\{[^{}]*\})", p.stdout)), key=lambda r: r["rank"])
    assert [r["rank"] for r in res] == [0, 1]
    # same target on both ranks (weights, mu), same number of chains, different chains
    assert res[0]["W0"] == res[1]["W0"] and res[0]["mu0"] == res[1]["mu0"]
    assert res[0]["n_chains"] == res[1]["n_chains"] == 64
    assert res[0]["theta_sum"] != res[1]["theta_sum"]
    # the slowest rank defines the step on every rank
    assert res[0]["ms"] == res[1]["ms"] == 15.0
    # rank-distinct random streams: rank r's chains are global chains r*B .. r*B + B - 1, so the
    # ranks' first normals differ while rank 0 reproduces the single-process stream
    assert [r["chain0"] for r in res] == [0, 64]
    assert res[0]["first"] != res[1]["first"]
    # the covariance-window exchange: both ranks hold rank 0's packet, then rank 1's
    assert res[0]["gathered"] == res[1]["gathered"] == [0.0, 1.0, 2.0, 3.0, 4.0, 100.0, 101.0, 102.0, 103.0, 104.0]
    from oracle import oracle as O
    assert res[0]["first"] == [float(x) for x in O.normals(7, 0, 0, 6)]
    assert res[1]["first"] == [float(x) for x in O.normals(7, 64, 0, 6)]


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "tiny_mala"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "tiny_mala"],
                       capture_output=True, text=True, timeout=300, env=env)
    import json
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
