"""Slab decomposition of a periodic grid over ranks.

The slowest axis (z in 3D, y in 2D) is cut into contiguous slabs, one per rank (one process per GPU).  Every rank
holds its planes plus one ghost plane at each end (`lbmk_grid_set_slab`).  After every collide-and-stream step the
only data another rank needs are the face-crossing populations of the two boundary planes (1 of Q directions per
face and component: nx*ny*m_total scalars per face):

    lbmk_halo_pack -> exchange with the two ring neighbours -> lbmk_halo_unpack

Overlap (the exchange "overlapped with the interior update"): `lbmk_step_slab` updates the two boundary
planes first, marks them with an event and then launches the interior planes; pack, transport and unpack run on a second
("comm") stream that waits for that event only, i.e. beside the interior launch; the next step waits for the unpack.
Same kernels and arithmetic as the serial order: the results are equal bit for bit (tests/test_gpu_slabs.py).

`HaloRing.exchange` is the transport: `torch.distributed` point-to-point (NCCL over NVLink on GPUs, gloo on CPU in
the tests) between ring neighbours, or plain copies when the ring has one rank.  This module only marshals buffers:
every step of the path, including packing and unpacking, runs in the kernels behind the C-ABI.
"""
from __future__ import annotations

from typing import List, Optional


class HaloRing:
    """Periodic ring of `world` ranks along the slab axis; rank r's lower neighbour is r-1, upper neighbour r+1."""

    def __init__(self, rank: int = 0, world: int = 1, dist=None):
        self.rank, self.world, self.dist = rank, world, dist
        self.lo = (rank - 1) % world
        self.hi = (rank + 1) % world
        if world > 1 and dist is None:
            raise ValueError("a ring of more than one rank needs torch.distributed")

    def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
        """recv_lo <- the lower neighbour's send_hi; recv_hi <- the upper neighbour's send_lo.

        world == 1: the rank is its own neighbour (periodic wrap through the ghost planes).
        world == 2: both neighbours are the same peer; messages between one pair of ranks are matched in posting
        order, so the receives are posted in the order the peer posts its sends (its send_lo, then its send_hi).
        """
        if self.world == 1:
            recv_lo.copy_(send_hi)
            recv_hi.copy_(send_lo)
            return
        d = self.dist
        if send_lo.is_cuda and d.get_backend() == "gloo":
            # gloo moves host memory only: stage through the host (the two-ranks-on-one-GPU test; NCCL takes the device buffers)
            h = [send_lo.cpu(), send_hi.cpu(), recv_hi.cpu(), recv_lo.cpu()]
            ops = [d.P2POp(d.isend, h[0], self.lo), d.P2POp(d.isend, h[1], self.hi),
                   d.P2POp(d.irecv, h[2], self.hi), d.P2POp(d.irecv, h[3], self.lo)]
            for req in d.batch_isend_irecv(ops):
                req.wait()
            recv_hi.copy_(h[2]); recv_lo.copy_(h[3])
            return
        ops = [d.P2POp(d.isend, send_lo, self.lo), d.P2POp(d.isend, send_hi, self.hi),
               d.P2POp(d.irecv, recv_hi, self.hi), d.P2POp(d.irecv, recv_lo, self.lo)]
        for req in d.batch_isend_irecv(ops):
            req.wait()


class SlabGrid:
    """One rank's slab of a periodic workload: a `Grid` in slab mode plus its four halo buffers."""

    def __init__(self, P, w_global, rank: int = 0, world: int = 1, device: str = "cuda:0", precision: Optional[str] = None):
        import torch
        import workloads as W
        self.torch = torch
        self.P = P
        self.rank, self.world = rank, world
        self.w = W.slab_workload(w_global, rank, world)
        self.start, self.count = W.slab_range(w_global.nz if w_global.dim == 3 else w_global.ny, world, rank)
        self.grid = P.Grid.from_workload(self.w, precision=precision, slab=True, device=device)
        m = self.w.m_total
        plane = self.w.nx * (self.w.ny if self.w.dim == 3 else 1)
        dt = torch.float64 if (precision or self.w.precision) in ("f64", "f64s") else torch.float32
        assert P.lbmk_halo_bytes(self.grid.h) == m * plane * (8 if dt == torch.float64 else 4)
        mk = lambda: torch.empty((m, plane), dtype=dt, device=self.grid.device)
        self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = mk(), mk(), mk(), mk()
        # halo pack / transport / unpack run on this stream, beside the interior update (None on a CPU stand-in grid: the
        # gloo test of the call order, tests/test_slabs_host.py)
        self.comm = torch.cuda.Stream(device=self.grid.device) if torch.device(self.grid.device).type == "cuda" else None

    def init(self):
        self.grid.init_from_U(self.w.initial_U())

    def pack(self):
        self.P.lbmk_halo_pack(self.grid.h, self.send_lo.data_ptr(), self.send_hi.data_ptr())

    def unpack(self):
        self.P.lbmk_halo_unpack(self.grid.h, self.recv_lo.data_ptr(), self.recv_hi.data_ptr())

    def step(self, n: int, ring: HaloRing, overlap: bool = True):
        """n steps, each with the halo exchange with the ring neighbours.  overlap: boundary planes first, then the
        exchange on the comm stream while the interior planes are updated on the grid's stream; otherwise step, pack,
        exchange, unpack in series on torch's current stream."""
        P, h, torch = self.P, self.grid.h, self.torch
        for _ in range(n):
            if not overlap:
                self.grid.step(1)
                self.pack()
                ring.exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi)
                self.unpack()
                continue
            self.begin_step()
            if self.comm is not None:
                with torch.cuda.stream(self.comm):
                    ring.exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi)
            else:
                ring.exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi)
            self.end_step()

    def begin_step(self):
        """Boundary planes, [event], interior planes on the grid's stream; pack on the comm stream after the event."""
        P, h, cs = self.P, self.grid.h, (self.comm.cuda_stream if self.comm is not None else 0)
        P.lbmk_step_slab(h)
        P.lbmk_stream_wait_boundary(h, cs)
        P.lbmk_halo_pack_on(h, self.send_lo.data_ptr(), self.send_hi.data_ptr(), cs)

    def end_step(self):
        """Unpack on the comm stream; the grid's stream (the next step) waits for it."""
        P, h, cs = self.P, self.grid.h, (self.comm.cuda_stream if self.comm is not None else 0)
        P.lbmk_halo_unpack_on(h, self.recv_lo.data_ptr(), self.recv_hi.data_ptr(), cs)
        P.lbmk_grid_wait_stream(h, cs)

    def read_U_interior(self):
        U = self.grid.read_U()
        return U[:, 1:-1] if self.w.dim == 3 else U[:, :, 1:-1]

    def close(self):
        self.grid.close()


def connect_local_peers(slabs: List[SlabGrid]):
    """Direct halo between slabs held by ONE process: every slab gets its ring neighbours' population buffers as peers
    (`lbmk_grid_set_halo_peers`).  Between GPUs the same pointers come from mapping the neighbour's workspace into this process
    (CUDA IPC / NVLink peer access): `connect_ipc_peers`."""
    P = slabs[0].P
    W = len(slabs)
    bufs = [P.lbmk_grid_population_buffers(s.grid.h) for s in slabs]
    for r, s in enumerate(slabs):
        lo, hi = bufs[(r - 1) % W], bufs[(r + 1) % W]
        P.lbmk_grid_set_halo_peers(s.grid.h, lo[0], lo[1], lo[2], hi[0], hi[1])


def connect_ipc_peers(slab: SlabGrid, ring: HaloRing):
    """Direct halo between RANKS (one process per GPU): every rank publishes its workspace through CUDA IPC (torch's storage
    sharing: cudaIpcGetMemHandle / cudaIpcOpenMemHandle, which also enables NVLink peer access), gathers its two ring neighbours'
    handles and registers their population buffers as halo peers.  Tested between two PROCESSES sharing one GPU
    (tests/test_gpu_slabs.py: same-device IPC mapping, gloo for the token); across GPUs (NVLink peer mapping, NCCL token) it is the
    same calls but has not run on this one-GPU pool.  Returns the mapped storages (keep them alive)."""
    torch, P, d = slab.torch, slab.P, ring.dist
    if ring.world == 1:
        connect_local_peers([slab])
        return []
    ws = slab.grid.workspace
    f0, f1, n0 = P.lbmk_grid_population_buffers(slab.grid.h)
    mine = dict(share=ws.untyped_storage()._share_cuda_(), base=ws.data_ptr(), f0=f0 - ws.data_ptr(), f1=f1 - ws.data_ptr(), n0=n0)
    everyone = [None] * ring.world
    d.all_gather_object(everyone, mine)
    keep, ptrs = [], []
    for peer in (ring.lo, ring.hi):
        info = everyone[peer]
        st = torch.UntypedStorage._new_shared_cuda(*info["share"])          # maps the peer's allocation into this process
        keep.append(st)
        # the handle covers the peer's whole cudaMalloc block; the tensor starts share[3] bytes into it
        base = st.data_ptr()
        ptrs.append((base + info["f0"], base + info["f1"], info["n0"]))
    P.lbmk_grid_set_halo_peers(slab.grid.h, ptrs[0][0], ptrs[0][1], ptrs[0][2], ptrs[1][0], ptrs[1][1])
    slab._tok = [torch.zeros(1, device=slab.grid.device) for _ in range(4)]
    return keep


def step_ring_peer(slab: SlabGrid, n: int, ring: HaloRing):
    """n steps of one rank with the direct halo (after `connect_ipc_peers`): the boundary launches store into the neighbours' ghost
    planes over NVLink while the interior launch runs; what goes through torch.distributed is a ONE-ELEMENT token per neighbour on
    the comm stream, sent after the boundary event: when the neighbour's token arrives, its peer stores have completed (stream
    order + kernel-boundary visibility), and the next step may read the ghost planes."""
    torch, P, h = slab.torch, slab.P, slab.grid.h
    t = slab._tok
    for _ in range(n):
        P.lbmk_step_slab_peer(h)
        P.lbmk_stream_wait_boundary(h, slab.comm.cuda_stream)
        with torch.cuda.stream(slab.comm):
            ring.exchange(t[0], t[1], t[2], t[3])
        P.lbmk_grid_wait_stream(h, slab.comm.cuda_stream)


def step_local_ring_peer(slabs: List[SlabGrid], n: int):
    """n steps of all slabs of a ring in one process with the direct halo: boundary planes (storing into the neighbours' ghost
    planes) -> interior; before its next step every slab's stream waits for both neighbours' boundary events."""
    P = slabs[0].P
    W = len(slabs)
    for _ in range(n):
        for s in slabs:
            P.lbmk_step_slab_peer(s.grid.h)
        for r, s in enumerate(slabs):
            cs = s.grid.stream.cuda_stream
            P.lbmk_stream_wait_boundary(slabs[(r - 1) % W].grid.h, cs)
            P.lbmk_stream_wait_boundary(slabs[(r + 1) % W].grid.h, cs)


def step_local_ring(slabs: List[SlabGrid], n: int, overlap: bool = False):
    """All slabs of a ring held by ONE process on one device (tests, and N = 1 with several slabs): every slab steps
    once, then the buffers are routed exactly as HaloRing.exchange routes them between ranks.  No kernel of one slab
    waits on another slab's kernel: the routing is plain stream-ordered copies."""
    W = len(slabs)
    if overlap:
        torch = slabs[0].torch
        for _ in range(n):
            for s in slabs:
                s.begin_step()
            for r, s in enumerate(slabs):           # each slab's comm stream takes its neighbours' packed buffers
                lo, hi = slabs[(r - 1) % W], slabs[(r + 1) % W]
                s.comm.wait_stream(lo.comm)
                s.comm.wait_stream(hi.comm)
                with torch.cuda.stream(s.comm):
                    s.recv_lo.copy_(lo.send_hi)
                    s.recv_hi.copy_(hi.send_lo)
            for r, s in enumerate(slabs):           # a neighbour's next pack must not overwrite a buffer still being copied
                slabs[(r - 1) % W].comm.wait_stream(s.comm)
                slabs[(r + 1) % W].comm.wait_stream(s.comm)
            for s in slabs:
                s.end_step()
        return
    for _ in range(n):
        for s in slabs:
            s.grid.step(1)
            s.pack()
        for r, s in enumerate(slabs):
            s.recv_lo.copy_(slabs[(r - 1) % W].send_hi)
            s.recv_hi.copy_(slabs[(r + 1) % W].send_lo)
        for s in slabs:
            s.unpack()
