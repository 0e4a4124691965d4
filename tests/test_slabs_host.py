"""Host side of the slab decomposition, on CPU: the split of the workload into slabs with
ghost planes, and the ring transport of `HaloRing.exchange` over torch.distributed `gloo` with world sizes 2 and 3
(world 2 is the case where both neighbours are the same peer)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("mk,kw,world", [(W.c4_nsf3d, dict(n=11, ny=6), 3), (W.c5_mhd3d, dict(n=7, ny=6), 2),
                                         (W.c2_swe, dict(n=13), 4), (W.c3_euler, dict(n=16), 3)])
def test_slab_workloads_tile_the_global_field_with_periodic_ghosts(mk, kw, world):
    # the slab axis must span the periodic unit box (n planes of spacing 1/n) for the analytic ghosts to wrap
    w = mk(**kw)
    U = w.initial_U()
    ax = 1 if w.dim == 3 else 2                       # slab axis in U[k][z][y][x]
    n_glob = U.shape[ax]
    covered = 0
    for r in range(world):
        start, count = W.slab_range(n_glob, world, r)
        assert start == covered
        covered += count
        ws = W.slab_workload(w, r, world)
        Us = ws.initial_U()
        assert Us.shape[ax] == count + 2
        idx = (np.arange(start - 1, start + count + 1)) % n_glob       # ghost planes = the neighbours' planes
        assert np.allclose(Us, np.take(U, idx, axis=ax), rtol=0, atol=1e-14)
    assert covered == n_glob


WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2607_05668_b200.slabs import HaloRing
dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ring = HaloRing(rank, world, dist)
out = []
for it in range(3):                                    # repeated exchanges stay matched
    send_lo = torch.full((4, 5), 100.0 * rank + 1 + 1000 * it)
    send_hi = torch.full((4, 5), 100.0 * rank + 2 + 1000 * it)
    recv_lo, recv_hi = torch.zeros(4, 5), torch.zeros(4, 5)
    ring.exchange(send_lo, send_hi, recv_lo, recv_hi)
    out.append([float(recv_lo[0, 0]), float(recv_hi[0, 0]), bool((recv_lo == recv_lo[0, 0]).all()), bool((recv_hi == recv_hi[0, 0]).all())])
dist.barrier()
print(json.dumps({{"rank": rank, "out": out}}))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


@pytest.mark.parametrize("world", [2, 3])
def test_halo_ring_exchange_gloo(world):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER.format(root=ROOT)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e
        d = json.loads(o.strip().splitlines()[-1])
        r = d["rank"]
        lo, hi = (r - 1) % world, (r + 1) % world
        for it, (rl, rh, ul, uh) in enumerate(d["out"]):
            assert ul and uh
            assert rl == 100.0 * lo + 2 + 1000 * it        # the lower neighbour's send_hi
            assert rh == 100.0 * hi + 1 + 1000 * it        # the upper neighbour's send_lo


def test_single_rank_ring_wraps_onto_itself():
    import torch
    from paper_2607_05668_b200.slabs import HaloRing
    a, b, rl, rh = torch.ones(2, 3), 2 * torch.ones(2, 3), torch.zeros(2, 3), torch.zeros(2, 3)
    HaloRing(0, 1).exchange(a, b, rl, rh)
    assert (rl == 2).all() and (rh == 1).all()
