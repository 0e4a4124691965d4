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


# ------------------------------------------------------------------------------------------------ SlabGrid.step end to end over gloo
# A CPU stand-in for the binding: the same calls SlabGrid makes (lbmk_step_slab, lbmk_stream_wait_boundary, lbmk_halo_pack[_on],
# lbmk_halo_unpack[_on], lbmk_grid_wait_stream, Grid.step) acting on a D2Q5 PURE-STREAMING state of integer tags in NumPy, with the
# library's halo protocol (send_lo = slot(-y) of the first own plane, send_hi = slot(+y) of the last own plane; recv_lo ->
# slot(+y) of the lower ghost plane, recv_hi -> slot(-y) of the upper ghost plane).  It records the call order.  What is tested is
# slabs.py: the order of calls in SlabGrid.step (overlapped and serial) and the routing between two ranks.
SLAB_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import workloads as W
from paper_2607_05668_b200.slabs import HaloRing, SlabGrid

C = [(0, 0), (1, 0), (-1, 0), (0, 1), (0, -1)]          # (cx, cy), direction order of include/lbmk.h

class FakeGrid:
    def __init__(self, w):
        self.w, self.h, self.device, self.log = w, self, torch.device("cpu"), []
        self.f = None
    def init_from_U(self, U):
        # tag populations: f_i = 10 * U + i (U carries the global node tag)
        self.f = np.stack([10.0 * U[0, 0] + i for i in range(5)])
    def _stream(self, rows):
        new = self.f.copy()
        for i, (cx, cy) in enumerate(C):
            src = np.roll(self.f[i], cx, axis=1)             # periodic in x inside the slab
            for y in rows:
                new[i, y] = src[y - cy]
        return new
    def step(self, n):
        assert n == 1
        self.log.append("step")
        self.f = self._stream(range(1, self.f.shape[1] - 1))

class FakeP:
    class Grid:
        @staticmethod
        def from_workload(w, precision=None, slab=False, device="cpu"):
            assert slab
            return FakeGrid(w)
    @staticmethod
    def lbmk_halo_bytes(g): return 1 * g.w.nx * 8
    @staticmethod
    def lbmk_step_slab(g):
        g.log.append("step_slab"); g.f = g._stream(range(1, g.f.shape[1] - 1))
    @staticmethod
    def lbmk_stream_wait_boundary(g, s): g.log.append("wait_boundary")
    @staticmethod
    def lbmk_grid_wait_stream(g, s): g.log.append("grid_wait_comm")
    @staticmethod
    def _pack(g, lo, hi):
        lo.copy_(torch.from_numpy(g.f[4, 1][None].copy())); hi.copy_(torch.from_numpy(g.f[3, -2][None].copy()))
    @staticmethod
    def _unpack(g, lo, hi):
        g.f[3, 0] = lo.numpy()[0]; g.f[4, -1] = hi.numpy()[0]

dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
nx, ny, steps = 6, 8, 5
tags = np.arange(nx * ny, dtype=np.float64).reshape(1, 1, ny, nx)
wg = W.relabel(W.c1_advection(nx, ny=ny), init=lambda w: tags[:, :, [(j + w.origin[1]) % ny for j in range(w.ny)], :].copy())
results = {{}}
for overlap in (True, False):
    s = SlabGrid(FakeP, wg, rank, world, device="cpu", precision="f64")
    # the binding hands device pointers; the stand-in needs the tensors themselves
    FakeP.lbmk_halo_pack = staticmethod(lambda g, a, b, s=s: (g.log.append("pack"), FakeP._pack(g, s.send_lo, s.send_hi)))
    FakeP.lbmk_halo_pack_on = staticmethod(lambda g, a, b, st, s=s: (g.log.append("pack_on"), FakeP._pack(g, s.send_lo, s.send_hi)))
    FakeP.lbmk_halo_unpack = staticmethod(lambda g, a, b, s=s: (g.log.append("unpack"), FakeP._unpack(g, s.recv_lo, s.recv_hi)))
    FakeP.lbmk_halo_unpack_on = staticmethod(lambda g, a, b, st, s=s: (g.log.append("unpack_on"), FakeP._unpack(g, s.recv_lo, s.recv_hi)))
    s.init()
    s.step(steps, HaloRing(rank, world, dist), overlap=overlap)
    results[str(overlap)] = dict(own=s.grid.f[:, 1:-1].tolist(), start=s.start, count=s.count, log=s.grid.log)
dist.barrier()
print(json.dumps(dict(rank=rank, res=results)))
dist.destroy_process_group()
"""


def test_slab_grid_step_over_gloo_world_2():
    """Two ranks, 5 steps, overlapped and serial: the slabs' own planes equal the global periodic streaming of the tags, and each
    step issues its calls in the documented order (boundary event before the pack; unpack before the grid's stream goes on)."""
    world, nx, ny, steps = 2, 6, 8, 5
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", SLAB_WORKER.format(root=ROOT)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    tags = np.arange(nx * ny, dtype=np.float64).reshape(ny, nx)
    C = [(0, 0), (1, 0), (-1, 0), (0, 1), (0, -1)]
    want = np.stack([np.roll(10.0 * tags + i, shift=(steps * cy, steps * cx), axis=(0, 1)) for i, (cx, cy) in enumerate(C)])
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-3000:]
        d = json.loads(o.strip().splitlines()[-1])
        for overlap in ("True", "False"):
            r = d["res"][overlap]
            own = np.array(r["own"])
            assert np.array_equal(own, want[:, r["start"]:r["start"] + r["count"]]), (d["rank"], overlap)
            per_step = (["step_slab", "wait_boundary", "pack_on", "unpack_on", "grid_wait_comm"] if overlap == "True"
                        else ["step", "pack", "unpack"])
            assert r["log"] == per_step * steps
