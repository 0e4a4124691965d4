#!/usr/bin/env python
"""bench.py -- MLUPS and achieved HBM GB/s of the fused collide-and-stream step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4] [--impl ours|reference]

A "step" is one collide-and-stream pass (eq 2.11; all rows a1-a7 of SURVEY.md §8(a)) over
the whole grid of the workload.  Default workload: BASELINE.json configs[3] ("c4": 3D compressible NSF with the
gradient-tracking cascade, 17 components, D3Q7, 256^3 periodic, shifted fp32, manufactured forcing on) -- the
larger of the two "3D fp32 configs" BASELINE.json's target is quoted on; it fits one GPU (8 GB per population
copy).  Inputs are the seeded synthetic fields of workloads/ (DESIGN.md "Input recipe").

One JSON line is printed by rank 0:
  value       MLUPS over all ranks, populations resident in HBM when the timed region starts
  e2e         the same metric through the public API with HOST buffers: lbmk_init_from_U(host U) -> K steps ->
              lbmk_read_U(host U), copies inside the timed region
  roofline    dominant kernel (collide_stream_*): algorithmic bytes 2*Q*m_total*sizeof per node (the byte model
              of the paper's Table 3) / CUDA-event time per launch, against the measured
              copy bandwidth in MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle (oracle/, plain fp64 C++) timed on this box's host cores on a bounded sample
  all_configs   short runs of the other BASELINE.json configs (reported, not the headline)
  paper_table3_systems  the paper's Table 3 systems compiled in here (4096^2, forcing off, S and D) next to the paper's
                RTX A5000 numbers (context); skipped with --no-table3 / --no-all-configs

Multi-GPU (--gpus N under torchrun): the path shards, so N > 1 runs SLABS by default -- ONE periodic grid
N times taller along the slowest axis, one workload-sized slab per rank, the face-crossing populations exchanged with the
ring neighbours after every step, overlapped with the interior update; value = node updates of all
ranks / max-over-ranks time; scaling "weak".  `--parallelism replicas` runs N independent full-size grids instead.

`--impl reference` times the oracle as it stands on host cores (rank 0 only): each step is one oracle step on a
bounded sub-box of the same workload (same node spacing and parameters), sized so the run ends within minutes.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "MLUPS (million lattice-node updates per second) of the fused collide-and-stream step"
UNIT = "MLUPS"

# dram__bytes_read.sum + dram__bytes_write.sum per collide_stream launch from the committed `ncu --set full`
# captures (profiles/), keyed by (config, pattern); None = not captured for this launch configuration.
NCU_TRAFFIC_BYTES = {}
try:
    with open(os.path.join(ROOT, "profiles", "traffic_per_launch.csv")) as _fh:
        for _ln in _fh.read().splitlines()[1:]:
            _k, _v = _ln.rsplit(",", 1)
            NCU_TRAFFIC_BYTES[_k] = int(_v)
except Exception:
    NCU_TRAFFIC_BYTES = {}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed LBM steps (default: the config's step count, capped at 200)")
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c4", choices=["c1", "c2", "c3", "c4", "c5", "hcnsf", "mhd2d", "swe_bathy"],
                    help="c1..c5: BASELINE.json configs; hcnsf (256^3), mhd2d, swe_bathy (4096^2): the paper's Table 3 systems added in "
                         "round 2, shifted fp32 (profiling targets, not headline workloads)")
    ap.add_argument("--pattern", default="auto", choices=["auto", "pull2", "aa"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "node", "twopass"])
    ap.add_argument("--n", "--edge", dest="n", type=int, default=None, help="override the grid edge (debug; the line then says so; --edge under torchrun, whose parser claims --n)")
    ap.add_argument("--no-mms", action="store_true", help="without manufactured forcing (the paper's Table 3 kernels carry none)")
    ap.add_argument("--stepping", default="auto", choices=["auto", "launch", "persistent", "cluster", "resident"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--parallelism", default="auto", choices=["auto", "replicas", "slabs"],
                    help="auto: slabs of one N-times-taller periodic grid with an overlapped halo exchange per step when N > 1; "
                         "replicas: N independent grids; slabs: force the slab path (also at N = 1, where the slab wraps onto itself)")
    ap.add_argument("--no-overlap", action="store_true", help="slabs: step, pack, exchange, unpack in series (no overlap)")
    ap.add_argument("--halo", default="nccl", choices=["nccl", "peer"],
                    help="slabs: nccl = pack / torch.distributed point-to-point / unpack beside the interior update (default, the "
                         "transport the CPU tests cover); peer = boundary kernels store straight into the neighbours' ghost planes "
                         "over CUDA-IPC-mapped peer memory, a one-element token for ordering (kernel tested on one GPU, the "
                         "cross-process wiring is not)")
    ap.add_argument("--backend", default="auto", choices=["auto", "nccl", "gloo"],
                    help="torch.distributed backend for N > 1 (auto: nccl); gloo + --one-device runs the N-rank path on ONE GPU (a dry "
                         "run of the multi-rank code path on pools with one GPU per call: halo buffers staged through the host)")
    ap.add_argument("--one-device", action="store_true", help="all ranks use cuda:0 (with --backend gloo)")
    ap.add_argument("--table3", action="store_true", help="(default on) also run the paper's Table 3 systems (4096^2, forcing off, S and D)")
    ap.add_argument("--no-table3", action="store_true")
    return ap.parse_args()


def make_workload(name, n=None, mms=True):
    import workloads as W
    kw = {}
    if n is not None:
        kw["n"] = n
    if name == "c4" and not mms:
        kw["mms"] = False
    if name in W.BASELINE_CONFIGS:
        w = W.BASELINE_CONFIGS[name](**kw)
    else:
        mk, n0 = {"hcnsf": (W.hcnsf3d, 256), "mhd2d": (W.pin_mhd2d, 4096), "swe_bathy": (W.pin_swe, 4096)}[name]
        w = W.relabel(mk(n or n0, precision="f32s"), steps=200)
    if not mms and w.mms_id:
        w = W.relabel(w, mms_id=0)
    return w


def measured_peak():
    """(GB/s, source) -- MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (torch copy, read+write bytes)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.perf_counter(), ln.strip()))

    def stop(self, t0=None, t1=None):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [ln for (t, ln) in self.lines if (t0 is None or t >= t0) and (t1 is None or t <= t1 + 0.06)] or [ln for _, ln in self.lines]
        for ln in rows:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); smax.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for nm, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


def dist_setup(n_gpus, backend="auto", one_device=False):
    """(rank, world, dist or None).  One process per GPU under torchrun; N = 1 needs no process group."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world == 1:
        return 0, 1, None
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if backend == "auto":
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    if torch.cuda.is_available():
        torch.cuda.set_device(0 if one_device else int(os.environ.get("LOCAL_RANK", "0")))
    dist.init_process_group(backend=backend)
    return rank, world, dist


def aggregate(dist, local_ms, local_node_updates, device="cpu"):
    """replicas-only aggregation: (max over ranks of the time, sum over ranks of the node updates)."""
    if dist is None:
        return local_ms, local_node_updates
    import torch
    if dist.get_backend() == "gloo":
        device = "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_node_updates)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def time_steps(g, torch, steps, dist=None):
    """CUDA-event time (ms) of exactly `steps` steps on the grid's stream, barrier + synchronize on both sides."""
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = g.launch_count()
    e0.record()
    g.step(steps)
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return e0.elapsed_time(e1), g.launch_count() - l0


class SlabRunner:
    """This rank's slab of the global workload behind the interface run_ours uses for a Grid."""

    def __init__(self, P, w_global, rank, world, dist, device, overlap=True, halo="nccl"):
        from paper_2607_05668_b200.slabs import HaloRing, SlabGrid
        self.overlap = overlap
        self.halo = halo
        self.slab = SlabGrid(P, w_global, rank, world, device=device)
        self.ring = HaloRing(rank, world, dist)
        self.grid = self.slab.grid
        self.w = self.slab.w                                   # local workload, ghost planes included
        self.pattern, self.kernel, self.shape_U = self.grid.pattern, self.grid.kernel, self.grid.shape_U
        plane = self.w.nx * (self.w.ny if self.w.dim == 3 else 1)
        self.own_nodes = plane * self.slab.count               # node updates that count: ghost planes excluded
        self._keep = None

    def init_from_U(self, U):
        self.grid.init_from_U(U)

    def step(self, n):
        if self.halo == "peer":
            from paper_2607_05668_b200.slabs import connect_ipc_peers, connect_local_peers, step_local_ring_peer, step_ring_peer
            if self._keep is None:
                self._keep = connect_ipc_peers(self.slab, self.ring)
            if self.ring.world == 1:
                step_local_ring_peer([self.slab], n)
            else:
                step_ring_peer(self.slab, n, self.ring)
            return
        self.slab.step(n, self.ring, overlap=self.overlap)

    def read_U(self, out=None):
        return self.grid.read_U(out)

    def max_wave_speed(self):
        return self.grid.max_wave_speed()

    def launch_count(self):
        return self.grid.launch_count()

    def close(self):
        self.slab.close()


def short_run(P, torch, name, pattern):
    """MLUPS / GB/s of one of the other configs (its full step count, 5% warm-up, median of 3).  L2-resident configs run
    launch-free (one cooperative launch per batch of steps, lbmk.h LBMK_STEPPING_PERSISTENT); the one-launch-per-step
    figure and, where one population copy fits the shared memory of all SMs, the SM-resident figure are reported beside it."""
    w = make_workload(name)
    out = None
    for stepping in ("auto", "launch", "resident"):
        g = P.Grid.from_workload(w, pattern=pattern if stepping != "resident" else "auto", stepping=stepping)
        if stepping != "auto" and (out["stepping"] == "launch" or g.stepping != stepping):      # large grids: one launch per step is all there is
            g.close()
            continue
        g.init_from_U(torch.from_numpy(w.initial_U()).cuda())
        g.step(max(10, w.steps // 20))
        reps, launches = [], 0
        for _ in range(3):
            ms, launches = time_steps(g, torch, w.steps)
            reps.append(ms)
        ms = statistics.median(reps)
        mlups = w.n_nodes * w.steps / (ms * 1e-3) / 1e6
        if out is None:
            out = {"workload": w.name, "dtype": "f64" if w.precision == "f64" else "f32", "pattern": g.pattern,
                   "stepping": g.stepping, "steps": w.steps, "launches": launches, "ms_per_step": ms / w.steps, "MLUPS": mlups,
                   "GBps_algorithmic": mlups * w.bytes_per_node / 1e3, "state_MB": w.n_nodes * w.bytes_per_node / 2 / 1e6}
        else:
            # "resident": LBMK_STEPPING_RESIDENT, one population copy in the shared memory of all SMs (AA pattern; opt-in)
            out["one_launch_per_step" if stepping == "launch" else "sm_resident"] = {"ms_per_step": ms / w.steps, "MLUPS": mlups, "launches": launches, "pattern": g.pattern}
        g.close()
    return out


# The paper's Table 3 rows that have a compiled-in system here: bulk collide-and-stream without
# manufactured forcing, single (shifted fp32) and double precision, on a saturating grid.  Paper columns: MLUPS and
# % of its 680 GB/s BabelStream peak on an RTX A5000 (context only -- another GPU, other kernels).
TABLE3 = [  # (label, workload maker name, paper S (MLUPS, %), paper D (MLUPS, %))
    ("burgers", "pin_burgers", (14474, 85.1), (7830, 92.1)),
    ("euler", "pin_euler", (4000, 94.1), (1003, 47.2)),
    ("swe", "c2_swe", (5093, 89.9), (958, 33.8)),
    ("ultrarelativistic", "pin_urf", (5349, 94.4), (1618, 57.1)),
    ("maxwell", "pin_maxwell", (5269, 93.0), (2634, 93.0)),
    ("adr", "pin_adr", (5405, 95.4), (1673, 59.0)),
    ("allen-cahn", "pin_allencahn", (5487, 96.8), (1918, 67.7)),
    ("incompressible-nse", "pin_inse", (2328, 95.8), (662, 54.6)),
    ("elasticity", "pin_elasticity", (2536, 89.5), (641, 45.2)),
    ("compressible-nsf", "pin_nsf2d", (1335, 94.2), (256, 36.2)),
    ("swe-bathymetry", "pin_swe", (5093, 89.9), (958, 33.8)),        # the same Table 3 row, with the bed-slope fields read per node
    ("resistive-mhd", "pin_mhd2d", (736, 78.0), (168, 35.7)),        # PAPER.md:L597-L598 (255 registers, spills there)
    ("hcnsf", "hcnsf3d", (546, 63.0), (163, 37.5)),                  # PAPER.md:L599-L600, D3Q7, 256^3 here
]


def table3_runs(P, torch, peak, n=4096, steps=40):
    """Our kernels on the paper's Table 3 systems: n x n periodic grid (state >> L2), forcing off, like the paper's."""
    import workloads as W
    out = {}
    for label, maker, paper_s, paper_d in TABLE3:
        for prec, paper in (("f32s", paper_s), ("f64", paper_d)):
            w = getattr(W, maker)(256 if maker == "hcnsf3d" else n, precision=prec)
            w = W.relabel(w, mms_id=0, steps=steps)
            try:
                g = P.Grid.from_workload(w)
                g.init_from_U(torch.from_numpy(w.initial_U()).cuda())
                g.step(5)
                ms = statistics.median(time_steps(g, torch, steps)[0] for _ in range(3))
                g.close()
                mlups = w.n_nodes * steps / (ms * 1e-3) / 1e6
                gbs = mlups * w.bytes_per_node / 1e3
                out[f"{label}:{'S' if prec == 'f32s' else 'D'}"] = {
                    "m_total": w.m_total, "n_prescribed_fields": w.n_aux, "bytes_per_node": w.bytes_per_node, "grid": [w.nx, w.ny, w.nz],
                    "MLUPS": mlups, "GBps_algorithmic": gbs,
                    "frac_of_measured_peak": gbs / peak, "paper_A5000_MLUPS": paper[0], "paper_pct_of_680GBps": paper[1]}
            except Exception as e:   # reported, never hidden
                out[f"{label}:{'S' if prec == 'f32s' else 'D'}"] = {"error": repr(e)}
            torch.cuda.empty_cache()
    return out


def cpu_baseline(w, budget_s=15.0):
    """The oracle as it stands on host cores, on a bounded sub-box of workload w (same dx, lambda, parameters)."""
    import numpy as np
    import oracle
    U0 = w.initial_U()
    # calibration box -> rate -> sample box
    def box(nz, ny):
        return (min(w.nz, nz) if w.dim == 3 else 1, min(w.ny, ny), w.nx)

    def run(bz, by, bx, steps):
        o = oracle.OracleGrid.from_workload(w, nx=bx, ny=by, nz=bz)
        o.init_from_U(np.ascontiguousarray(U0[:, :bz, :by, :bx]))
        o.step(1)
        t = time.perf_counter()
        o.step(steps)
        dt = time.perf_counter() - t
        o.close()
        return bz * by * bx * steps / dt / 1e6, dt

    bz, by, bx = box(4, 64)
    rate, _ = run(bz, by, bx, 2)
    target_updates = rate * 1e6 * budget_s
    steps = 8
    plane = w.nx * w.ny
    if w.dim == 3:
        bz = int(max(4, min(w.nz, target_updates / steps / plane)))
        by = w.ny
    else:
        bz, by = 1, int(max(8, min(w.ny, target_updates / steps / w.nx)))
        steps = int(max(8, min(w.steps, target_updates / (by * w.nx))))
    mlups, dt = run(bz, by, w.nx, steps)
    return {"value": mlups, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle",
            "sample": f"{steps} steps (after 1 warm-up) on a periodic {w.nx}x{by}x{bz} sub-box of {w.name} "
                      f"(same dx, lambda, parameters, forcing); {dt:.1f} s wall"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np
    import oracle
    w = make_workload(args.config, args.n, not args.no_mms)
    steps = args.steps if args.steps is not None else min(w.steps, 200)
    warm = args.warmup
    U0 = w.initial_U()
    # calibrate on a tiny box, then size the sample so (steps + warm) oracle steps take about two minutes
    cz, cy = (4 if w.dim == 3 else 1), min(w.ny, 64)
    o = oracle.OracleGrid.from_workload(w, nx=w.nx, ny=cy, nz=cz)
    o.init_from_U(np.ascontiguousarray(U0[:, :cz, :cy, :]))
    o.step(1)
    t = time.perf_counter(); o.step(2); rate = cz * cy * w.nx * 2 / (time.perf_counter() - t)
    o.close()
    per_step = rate * 120.0 / (steps + warm)
    if w.dim == 3:
        by = w.ny
        bz = int(max(2, min(w.nz, per_step / (w.nx * w.ny))))
        if bz == 2:
            by = int(max(8, min(w.ny, per_step / (w.nx * bz))))
    else:
        bz, by = 1, int(max(8, min(w.ny, per_step / w.nx)))
    o = oracle.OracleGrid.from_workload(w, nx=w.nx, ny=by, nz=bz)
    o.init_from_U(np.ascontiguousarray(U0[:, :bz, :by, :]))
    o.step(warm)
    t = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t
    o.close()
    nodes = bz * by * w.nx
    mlups = nodes * steps / dt / 1e6
    sample = f"each step = one oracle step on a periodic {w.nx}x{by}x{bz} sub-box of {w.name} (same dx, lambda, parameters, forcing)"
    line = {"impl": "reference", "metric": METRIC, "value": mlups, "unit": UNIT, "n_gpus": args.gpus, "steps": steps, "warmup": warm,
            "ms_per_step": dt * 1e3 / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": w.name, "system": w.system, "lattice": w.lattice, "m_total": w.m_total,
                                            "grid": [w.nx, w.ny, w.nz], "sample_grid": [w.nx, by, bz], "note": sample},
            "cpu_baseline": {"value": mlups, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": mlups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import numpy as np
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the collide-and-stream path has no CPU fallback "
                         "(use --impl reference for the CPU oracle)")
    rank, world, dist = dist_setup(args.gpus, args.backend, args.one_device)
    local = 0 if args.one_device else int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    import paper_2607_05668_b200 as P
    P.lib()

    w = make_workload(args.config, args.n, not args.no_mms)
    steps = args.steps if args.steps is not None else min(w.steps, 200)
    warm = max(args.warmup, 3)
    dev = f"cuda:{local}"
    slabs = args.parallelism == "slabs" or (args.parallelism == "auto" and world > 1)
    if slabs:
        import workloads as W
        # weak scaling: one periodic grid `world` times taller along the slab axis, this rank owns one workload-sized slab
        wg = W.relabel(w, **({"nz": w.nz * world} if w.dim == 3 else {"ny": w.ny * world}))
        g = SlabRunner(P, wg, rank, world, dist, dev, overlap=not args.no_overlap, halo=args.halo)
        own_nodes, U0 = g.own_nodes, g.w.initial_U()
    else:
        own_nodes, U0 = w.n_nodes, w.initial_U()
        g = P.Grid.from_workload(w, pattern=args.pattern, kernel=args.kernel, stepping=args.stepping, device=dev)
    U0_dev = torch.from_numpy(U0).to(dev)
    g.init_from_U(U0_dev)
    speeds, status = g.max_wave_speed()                      # a10: device sub-characteristic check (untimed)
    g.step(warm)
    sampler = ClockSampler(local).start() if rank == 0 else None
    # keep the sampler busy for a while before the timed region so that it has samples
    t_wall0 = time.perf_counter()
    reps = []
    n_rep = 3
    launches = 0
    for _ in range(n_rep):
        ms, launches = time_steps(g, torch, steps, dist)
        reps.append(ms)
    t_wall1 = time.perf_counter()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms_local = statistics.median(reps)
    ms, updates = aggregate(dist, ms_local, own_nodes * steps, dev)
    mlups = updates / (ms * 1e-3) / 1e6
    finite = bool(np.isfinite(g.read_U(torch.empty(g.shape_U, dtype=torch.float64, device=dev)).sum().item()))

    # e2e through the public API with host buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        U_host = torch.from_numpy(U0).pin_memory()
        out_host = torch.empty(g.shape_U, dtype=torch.float64).pin_memory()
        g.init_from_U(U_host); g.step(2); g.read_U(out_host)      # warm the staging pool
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tw = time.perf_counter()
        e0.record()
        g.init_from_U(U_host)
        g.step(steps)
        g.read_U(out_host)
        e1.record()
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - tw) * 1e3
        e_ms = max(e0.elapsed_time(e1), wall_ms)
        e_ms, e_upd = aggregate(dist, e_ms, own_nodes * steps, dev)
        nbytes = U_host.numel() * 8
        e2e = {"value": e_upd / (e_ms * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": nbytes / steps,
               "d2h_bytes_per_step": nbytes / steps, "ms_total": e_ms,
               "what": f"lbmk_init_from_U(pinned host U, {nbytes / 1e6:.0f} MB) -> {steps} steps -> lbmk_read_U(pinned host)"}
        del U_host, out_host
    pattern, kernel, mode = g.pattern, g.kernel, getattr(g, "stepping", "launch")
    g.close()
    del g, U0_dev
    torch.cuda.empty_cache()

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    peak, peak_src = measured_peak()
    # the library's own streaming probe (plain float4 copy kernel, read + write bytes), cf. the paper's BabelStream peak
    try:
        nb = 1 << 30
        a_, b_ = torch.empty(nb, dtype=torch.uint8, device=dev), torch.empty(nb, dtype=torch.uint8, device=dev)
        P.lbmk_copy_bandwidth(b_.data_ptr(), a_.data_ptr(), nb, 3, torch.cuda.current_stream().cuda_stream)
        probe = P.lbmk_copy_bandwidth(b_.data_ptr(), a_.data_ptr(), nb, 10, torch.cuda.current_stream().cuda_stream)
        del a_, b_
    except Exception as e:   # reported, never hidden
        probe = repr(e)
    bytes_per_launch = w.n_nodes * w.bytes_per_node
    ms_launch = ms_local / steps
    achieved = bytes_per_launch / (ms_launch * 1e-3) / 1e9
    # persistent / cluster / resident launches have their own captures (per step)
    key = f"{args.config}:{pattern}:{kernel}" + ("" if mode == "launch" else f":{mode}")
    traffic = NCU_TRAFFIC_BYTES.get(key) if args.n is None else None    # captured at the full size only
    line = {
        "metric": METRIC, "value": mlups, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
        "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if w.precision == "f64" else "f32", "data": "synthetic",
        "config": {"workload": w.name, "system": w.system, "lattice": w.lattice, "m_conserved": None, "m_total": w.m_total,
                   "grid": [w.nx, w.ny, w.nz], "precision": w.precision, "mms_forcing": bool(w.mms_id),
                   "pattern": pattern, "kernel": kernel, "bytes_per_node": w.bytes_per_node,
                   "l2": "state larger than L2 (no flush needed)" if bytes_per_launch / 2 > 2.5e8 else "state fits in L2: HBM roofline n/a",
                   "parallelism": (("slabs along the slowest axis, " + ("boundary kernels store into the neighbours' ghost planes over peer memory" if args.halo == "peer" else "halo exchange per step" + (" overlapped with the interior update" if not args.no_overlap else ", serial")))
                                   if slabs else "replicas only") if (world > 1 or slabs) else "single GPU", "timing": f"median of {n_rep} x {steps} steps, CUDA events",
                   "lattice_wave_speed": max(speeds[0], speeds[1]) + speeds[2], "finite": finite},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic,
                     "traffic_source": ("constant from profiles/traffic_per_launch.csv: dram__bytes_read.sum + dram__bytes_write.sum of one "
                                        "`ncu --set full` capture of this kernel and launch configuration (profiles/), NOT measured by this run")
                                       if traffic is not None else None,
                     "peak_source": peak_src, "frac_of_nominal_8TBps": achieved / 8000.0,
                     "kernel": {"launch": "collide_stream_node (one launch per step)",
                                "persistent": "collide_stream_persistent (one cooperative launch per lbmk_step call; figures per step)",
                                "cluster": "collide_stream_cluster (one cluster launch per lbmk_step call; figures per step)",
                                "resident": "collide_stream_resident (state in the shared memory of all SMs, one cooperative launch per lbmk_step call; figures per step)"}.get(
                                    mode, "collide_stream"),
                     "stepping": mode, "algorithmic_bytes_per_launch": bytes_per_launch,
                     "lbmk_copy_probe_GBps": probe,
                     "frac_of_max_measured_copy": achieved / max(peak, probe) if isinstance(probe, float) else None},
        "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
    }
    line["config"].pop("m_conserved")
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(w)
    if not args.no_all_configs and world == 1:
        others = {}
        for name in ("c1", "c2", "c3", "c4", "c5"):
            if name == args.config:
                continue
            try:
                r = short_run(P, torch, name, args.pattern)
                r["frac_of_measured_peak"] = r["GBps_algorithmic"] / peak
                others[name] = r
            except Exception as e:   # reported, never hidden
                others[name] = {"error": repr(e)}
            torch.cuda.empty_cache()
        line["all_configs"] = others
    if not args.no_table3 and not args.no_all_configs and world == 1 or args.table3 and world == 1:
        line["paper_table3_systems"] = table3_runs(P, torch, peak)
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
