"""Slab decomposition on the device: several slabs of one periodic grid, held by one process
on one GPU and exchanged exactly as the ranks of a ring exchange them, reproduce the single-grid run BIT FOR BIT
(same kernels, same arithmetic; the ghost planes and halo pack/unpack are the only difference)."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2607_05668_b200 as P
    P.lib()
    return P


# the slab axis spans the periodic unit box (n planes), so that the analytic ghost planes wrap
CASES = [(W.pin_swe, dict(n=24), 3, 9), (W.hcnsf3d, dict(n=10, ny=6), 2, 6),      # systems with prescribed per-node fields
         (W.c4_nsf3d, dict(n=13, ny=10), 3, 9), (W.c4_nsf3d, dict(n=128, ny=4, precision="f64"), 2, 5),
         (W.c5_mhd3d, dict(n=9, ny=10), 4, 8), (W.c2_swe, dict(n=17), 3, 11), (W.c2_swe, dict(n=256), 2, 6),
         (W.c3_euler, dict(n=32), 2, 10), (W.pin_adr, dict(n=16), 3, 12)]


@pytest.mark.parametrize("overlap", [False, True, "peer"])
@pytest.mark.parametrize("mk,kw,world,steps", CASES)
def test_slabs_reproduce_the_single_grid_bit_for_bit(P, mk, kw, world, steps, overlap):
    from paper_2607_05668_b200.slabs import SlabGrid, step_local_ring
    w = mk(**kw)
    g = P.Grid.from_workload(w, pattern="pull2")
    g.init_from_U(w.initial_U())
    g.step(steps)
    U = g.read_U()
    speeds = g.max_wave_speed()[0]
    norms = P.lbmk_error_norms(g.h, w.m_total) if w.mms_id else None      # raw sums / maxima
    g.close()
    slabs = [SlabGrid(P, w, r, world) for r in range(world)]
    for s in slabs:
        s.init()
    if overlap == "peer":                              # compute + halo in one kernel: boundary blocks store into the neighbours' ghost planes
        from paper_2607_05668_b200.slabs import connect_local_peers, step_local_ring_peer
        connect_local_peers(slabs)
        step_local_ring_peer(slabs, steps)
    else:
        step_local_ring(slabs, steps, overlap=overlap)     # overlap: boundary planes first, exchange beside the interior update
    ax = 1 if w.dim == 3 else 2
    Us = np.concatenate([s.read_U_interior() for s in slabs], axis=ax)
    assert Us.shape == U.shape
    if overlap == "peer":
        # the boundary planes are updated by the peer-store instantiation of the step kernel: same arithmetic, but nvcc decides FMA
        # contraction per kernel, so nonlinear systems agree to rounding (linear ones bit for bit); the transfer itself is exact
        scale = np.abs(U).max()                       # system scale: short runs hold components that have barely left zero
        assert np.abs(Us - U).max() / scale <= (1e-13 if w.precision == "f64" else 1e-6)
        for s in slabs:
            s.close()
        return
    assert np.array_equal(Us, U)
    # the reductions skip the ghost planes: max over slabs = the single grid's value
    sp = np.max([s.grid.max_wave_speed()[0] for s in slabs], axis=0)
    assert np.allclose(sp, speeds, rtol=1e-14)
    if norms is not None:
        parts = [P.lbmk_error_norms(s.grid.h, w.m_total) for s in slabs]
        for j in (0, 1, 3, 4):                               # sums add up over the slabs
            assert np.allclose(sum(p[:, j] for p in parts), norms[:, j], rtol=1e-12, atol=1e-300)
        for j in (2, 5):                                     # maxima: max over the slabs
            assert np.array_equal(np.max([p[:, j] for p in parts], axis=0), norms[:, j])
    for s in slabs:
        s.close()


@pytest.mark.parametrize("overlap", [False, True])
def test_one_rank_ring_equals_periodic_grid(P, overlap):
    """world = 1: the slab's ghost planes wrap onto the slab itself through HaloRing.exchange."""
    from paper_2607_05668_b200.slabs import HaloRing, SlabGrid
    w = W.c5_mhd3d(n=10, ny=8)
    g = P.Grid.from_workload(w, pattern="pull2")
    g.init_from_U(w.initial_U())
    g.step(7)
    U = g.read_U()
    g.close()
    s = SlabGrid(P, w, 0, 1)
    s.init()
    s.step(7, HaloRing(0, 1), overlap=overlap)
    assert np.array_equal(s.read_U_interior(), U)
    s.close()


def test_halo_calls_are_refused_out_of_order(P):
    w = W.c5_mhd3d(n=6)
    g = P.Grid.from_workload(w)                              # not a slab
    g.init_from_U(w.initial_U()); g.step(1)
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_halo_pack(g.h, g.workspace.data_ptr(), g.workspace.data_ptr())
    assert e.value.status == 5
    g.close()
    s = P.Grid.from_workload(W.slab_workload(w, 0, 2), slab=True)
    s.init_from_U(W.slab_workload(w, 0, 2).initial_U())
    with pytest.raises(P.LbmkError) as e:                    # before the first step: ghosts come from init
        P.lbmk_halo_pack(s.h, s.workspace.data_ptr(), s.workspace.data_ptr())
    assert e.value.status == 5 and s.pattern == "pull2"
    s.close()



def test_peer_halo_calls_are_refused_out_of_order(P):
    w = W.c5_mhd3d(n=6)
    ws = W.slab_workload(w, 0, 2)
    s = P.Grid.from_workload(ws, slab=True)
    s.init_from_U(ws.initial_U())
    with pytest.raises(P.LbmkError) as e:                    # no peers registered
        P.lbmk_step_slab_peer(s.h)
    assert e.value.status == 5
    f0, f1, n0 = P.lbmk_grid_population_buffers(s.h)
    assert f0 and f1 and f1 != f0 and n0 == (ws.nz - 1) * ws.nx * ws.ny
    with pytest.raises(P.LbmkError):
        P.lbmk_grid_set_halo_peers(s.h, 0, f1, n0, f0, f1)   # NULL peer buffer
    s.close()
    t = P.Grid.from_workload(ws, slab=True, collision="trt")
    t.init_from_U(ws.initial_U())
    f0, f1, n0 = P.lbmk_grid_population_buffers(t.h)
    P.lbmk_grid_set_halo_peers(t.h, f0, f1, n0, f0, f1)
    with pytest.raises(P.LbmkError) as e:                    # the peer-store instantiation exists for BGK only
        P.lbmk_step_slab_peer(t.h)
    assert e.value.status == 6
    t.close()
    g = P.Grid.from_workload(w)
    with pytest.raises(P.LbmkError) as e:                    # not a slab
        P.lbmk_grid_set_halo_peers(g.h, f0, f1, 0, f0, f1)
    assert e.value.status == 5
    g.close()


TWO_RANK_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import paper_2607_05668_b200 as P, workloads as W
from paper_2607_05668_b200.slabs import HaloRing, SlabGrid, connect_ipc_peers, step_ring_peer
dist.init_process_group(backend="gloo")               # NCCL refuses two ranks on one GPU; gloo moves the same CUDA buffers
rank, world = dist.get_rank(), dist.get_world_size()
w = W.c5_mhd3d(n=10, ny=8)
out = {{}}
for overlap in (True, False):
    s = SlabGrid(P, w, rank, world, device="cuda:0")
    s.init()
    s.step(6, HaloRing(rank, world, dist), overlap=overlap)
    out[str(overlap)] = s.read_U_interior().tolist()
    s.close()
# direct halo: each rank maps the other's workspace through CUDA IPC and its boundary kernels store into the other's ghost planes
s = SlabGrid(P, w, rank, world, device="cuda:0")
s.init()
ring = HaloRing(rank, world, dist)
keep = connect_ipc_peers(s, ring)
step_ring_peer(s, 6, ring)
out["peer"] = s.read_U_interior().tolist()
dist.barrier()
del keep
s.close()
dist.barrier()
print(json.dumps(dict(rank=rank, start=s.start, count=s.count, out=out)))
dist.destroy_process_group()
"""


def test_two_ranks_on_one_gpu_over_gloo_reproduce_the_single_grid(P):
    """The multi-process path end to end with real kernels: two RANKS (processes), one slab each, both on this one GPU, the halo
    buffers moved by torch.distributed point-to-point (gloo here, because NCCL needs one GPU per rank; the calls are the ones the
    NCCL run makes).  No kernel of one rank waits on a kernel of the other: ordering is host-side.  Overlapped and serial, and
    the direct halo: the ranks map each other's workspace through CUDA IPC (`connect_ipc_peers`) and the boundary kernels store
    into the other PROCESS's ghost planes, a one-element token per neighbour for ordering (`step_ring_peer`)."""
    import json, os, socket, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    w = W.c5_mhd3d(n=10, ny=8)
    g = P.Grid.from_workload(w, pattern="pull2")
    g.init_from_U(w.initial_U()); g.step(6)
    U = g.read_U(); g.close()
    sk = socket.socket(); sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]; sk.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", TWO_RANK_WORKER.format(root=root)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    for p in procs:
        try:
            o, e = p.communicate(timeout=240)
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            raise
        assert p.returncode == 0, e[-3000:]
        d = json.loads(o.strip().splitlines()[-1])
        for overlap in ("True", "False"):
            own = np.array(d["out"][overlap])
            assert np.array_equal(own, U[:, d["start"]:d["start"] + d["count"]]), (d["rank"], overlap)
        own = np.array(d["out"]["peer"])              # CUDA-IPC peer stores between the two processes: equal to rounding (fp32 here)
        assert np.abs(own - U[:, d["start"]:d["start"] + d["count"]]).max() <= 1e-6 * np.abs(U).max(), d["rank"]


@pytest.mark.parametrize("halo", ["nccl", "peer"])
def test_bench_multi_rank_path_dry_run_on_one_gpu(P, halo):
    """`bench.py --gpus 2` as the driver launches it (torch.distributed.run, one process per rank), but with both ranks on this one
    GPU and gloo as transport: the slab default for N > 1, max-over-ranks timing, sum-over-ranks node updates, rank 0 prints ONE
    JSON line.  A dry run of the code path, not a measurement."""
    import json, os, socket, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sk = socket.socket(); sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]; sk.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "6", "--warmup", "3",
           "--backend", "gloo", "--one-device", "--edge", "32", "--halo", halo, "--no-cpu-baseline"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=400, cwd=root)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["steps"] == 6 and d["scaling"] == "weak" and d["config"]["finite"] is True
    assert d["config"]["parallelism"].startswith("slabs") and d["value"] > 0 and d["gpu_launches"] >= 6
