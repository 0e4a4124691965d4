"""N > 1 path of bench.py on CPU: world-size-2 `gloo` run of the replicas-only aggregation.

Each rank reports its own CUDA-event time and node updates; the job value is sum(updates) / max(time).  The test
runs bench.dist_setup + bench.aggregate in two real processes over gloo (rendezvous on 127.0.0.1) and checks the
max / sum semantics and that the `--impl reference` leg stays silent on ranks != 0.
"""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import bench
rank, world, dist = bench.dist_setup(2)
assert world == 2 and dist is not None and dist.get_backend() == "gloo"
ms, upd = bench.aggregate(dist, 10.0 + 5.0 * rank, 1000 * (rank + 1))
dist.barrier()
print(json.dumps({{"rank": rank, "ms": ms, "updates": upd}}))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_replicas_aggregate_world_size_2_gloo():
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER.format(root=ROOT)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=120) for p in procs]
    import json
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
        d = json.loads(o.strip().splitlines()[-1])
        assert d["ms"] == 15.0          # max over ranks
        assert d["updates"] == 3000.0   # sum over ranks


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
