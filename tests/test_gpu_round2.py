"""GPU tests of what round 2 added to the path (all through the C-ABI):
  * launch-free stepping: the persistent cooperative kernel equals the per-launch path BIT FOR BIT;
  * prescribed per-node coefficient fields (bed slope of eq 3.5): shallow water over a bed and
    the homogenized NSF system (eq 3.27), element by element against the oracle;
  * resistive MHD 2D with the Powell source (eq 3.25; 18 fields), against the oracle;
  * node-range launches (the slab's boundary / interior split).
"""
import numpy as np
import pytest

import oracle
import workloads as W
from parity_metric import gate

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m 'not gpu' on CPU boxes)")
    import paper_2607_05668_b200 as P
    P.lib()
    return P


def gpu_run(P, w, steps, chunks=None, **kw):
    g = P.Grid.from_workload(w, **kw)
    g.init_from_U(w.initial_U())
    for c in (chunks or [steps]):
        g.step(c)
    assert g.time()[0] == steps
    U, f = g.read_U(), g.read_populations()
    info = (g.stepping, g.launch_count())
    g.close()
    return U, f, info


def oracle_run(w, steps, aux_in_time=False):
    o = oracle.OracleGrid.from_workload(w)
    if o.n_aux:
        o.set_aux(w.aux_fields(0.0))
    o.init_from_U(w.initial_U())
    if aux_in_time:
        for s in range(steps):
            o.set_aux(w.aux_fields((s + 0.5) * w.dt))        # explicit (x, t) dependence at the midpoint
            o.step(1)
    else:
        o.step(steps)
    Uo, fo = o.read_U(), o.read_f()
    o.close()
    return Uo, fo


# ------------------------------------------------------------------------------------------- persistent stepping
PERSIST = [
    (W.c1_advection, dict(n=64), 200, None),                        # configs[0] at full size and duration
    (W.c1_advection, dict(n=37, ny=23), 51, [1, 2, 48]),            # ragged, odd chunks (first chunk is the LOCAL step)
    (W.c2_swe, dict(n=128, ny=40), 150, [70, 1, 79]),               # forcing on, staged row coefficients, > 2 coefficient batches
    (W.c2_swe, dict(n=96, ny=50), 67, None),                        # forcing on, unstaged (nx not a multiple of the block)
    (W.c3_euler, dict(n=80, ny=36), 61, None),                      # shifted fp32
    (W.c4_nsf3d, dict(n=64, ny=6, nz=5), 30, None),                 # 17 fields, fp32, forcing on, staged (nx = block)
    (W.c5_mhd3d, dict(n=24, ny=10, nz=7, precision="f64"), 31, None),
    (W.pin_swe, dict(n=40), 50, None),                              # prescribed per-node fields
    (lambda: W.relabel(W.pin_burgers(88), mms_id=0), dict(), 40, [3, 37]),     # 7744 nodes, no forcing: the largest cluster-resident class (npc = 992)
    (lambda: W.relabel(W.c2_swe(72, ny=50), mms_id=0), dict(), 45, [2, 43]),  # SWE without forcing: cluster-resident, fp64, nonlinear
]


@pytest.mark.parametrize("mk,kw,steps,chunks", PERSIST)
def test_persistent_stepping_is_bit_identical_to_per_launch(P, mk, kw, steps, chunks):
    """SURVEY.md section 7 "Small configs": one cooperative launch per batch of steps with a grid barrier between steps runs the
    same per-node code (kernels.cuh node_step) as the one-launch-per-step path, so the populations agree bit for bit."""
    w = mk(**kw)
    U1, f1, (mode1, l1) = gpu_run(P, w, steps, chunks, pattern="pull2", stepping="launch")
    U2, f2, (mode2, l2) = gpu_run(P, w, steps, chunks, pattern="pull2", stepping="persistent")
    assert mode1 == "launch" and mode2 == "persistent"
    assert np.array_equal(f1, f2) and np.array_equal(U1, U2)
    assert l2 < l1                                                  # fewer launches is the point
    Uo, fo = oracle_run(w, steps)
    gate(U2, Uo, fo, w.precision, f"{w.name}[persistent]", U_ref=w.U_ref, steps=steps, strict=False)
    # cluster-resident kernel (state in distributed shared memory): same arithmetic (collide_core), FMA contraction decided per
    # kernel by nvcc -> equal to rounding in general, bit for bit for the linear system of configs[0]
    U3, f3, (mode3, l3) = gpu_run(P, w, steps, chunks, pattern="pull2", stepping="cluster")
    if mode3 == "cluster":
        assert l3 <= l2
        if w.system == "advection2d":
            assert np.array_equal(f1, f3)
        d = np.abs(f3 - f1).max() / np.abs(f1).max()
        assert d <= (2e-7 if w.precision == "f32s" else 1e-13), d
        gate(U3, Uo, fo, w.precision, f"{w.name}[cluster]", U_ref=w.U_ref, steps=steps, strict=False)
    else:
        assert mode3 == "persistent" and np.array_equal(f1, f3)     # does not qualify: falls back


RESIDENT = PERSIST + [
    (W.c2_swe, dict(n=512, ny=40), 33, [1, 32]),                    # 160 tiles over 148 SMs: 2 tiles per block, every tile a boundary tile
    (W.c2_swe, dict(n=200, ny=301), 21, [2, 19]),                   # 60 200 nodes: tiles straddle rows, ragged last tile, interior tiles exist
    (W.hcnsf3d, dict(n=20, ny=18, nz=16), 12, [5, 7]),              # 3D, prescribed fields, reach = nx*ny
    (W.c4_nsf3d, dict(n=24, ny=20, nz=18), 9, None),                # 3D, 17 fields, forcing on
]


@pytest.mark.parametrize("mk,kw,steps,chunks", RESIDENT)
def test_sm_resident_stepping_is_bit_identical_to_aa_per_launch(P, mk, kw, steps, chunks):
    """LBMK_STEPPING_RESIDENT: every block keeps its tiles in shared memory (global layout, AA pattern in place), only block-boundary
    populations stay in global memory, neighbouring blocks synchronised by step flags.  The arithmetic is collide_core: the
    populations agree bit for bit with the per-launch AA path -- odd and even step counts, calls starting at either AA parity."""
    w = mk(**kw)
    U1, f1, (mode1, l1) = gpu_run(P, w, steps, chunks, pattern="aa", stepping="launch")
    U2, f2, (mode2, l2) = gpu_run(P, w, steps, chunks, stepping="resident")
    assert mode1 == "launch" and mode2 == "resident"
    if w.mms_id and w.system in ("nsf3d", "nsf2d", "inse2d", "mhd2d"):
        # >= 48 row coefficients: the per-launch kernel may read them from its shared-memory copy, the resident kernel reads global
        # memory -- two instantiations of the forcing polynomial, equal to rounding
        d = np.abs(f2 - f1).max() / np.abs(f1).max()
        assert d <= (1e-6 if w.precision == "f32s" else 1e-13), d
    else:
        assert np.array_equal(f1, f2) and np.array_equal(U1, U2)
    assert l2 < l1
    Uo, fo = oracle_run(w, steps)
    gate(U2, Uo, fo, w.precision, f"{w.name}[resident]", U_ref=w.U_ref, steps=steps, strict=False)


def test_sm_resident_stepping_falls_back_when_the_grid_does_not_fit(P):
    w = W.c3_euler(n=1024, precision="f32s")                        # 1M nodes x 80 B = 84 MB: more than all shared memory together
    g = P.Grid.from_workload(w, stepping="resident")
    assert g.pattern == "aa" and g.stepping == "launch"
    g.close()
    g = P.Grid.from_workload(W.c2_swe(), stepping="resident")       # configs[1]: 31 MB, 14 tiles (215 KB) per SM
    assert (g.pattern, g.stepping) == ("aa", "resident")
    g.close()
    g = P.Grid.from_workload(W.c2_swe(n=64), stepping="resident", pattern="pull2")    # an explicit two-lattice pattern wins
    assert (g.pattern, g.stepping) == ("pull2", "persistent")
    g.close()


def test_persistent_is_the_default_for_l2_resident_grids_only(P):
    tiny = P.Grid.from_workload(W.c1_advection())                   # configs[0]: 4096 nodes, no forcing -> one cluster, DSMEM-resident
    assert tiny.stepping == "cluster"
    tiny.close()
    small = P.Grid.from_workload(W.c2_swe(64))                      # forcing on -> cooperative persistent kernel
    assert small.stepping == "persistent"
    small.close()
    aa = P.Grid.from_workload(W.c2_swe(64), pattern="aa")           # in-place pattern: per-launch only
    assert aa.stepping == "launch"
    aa.close()
    big = P.Grid.from_workload(W.c3_euler(2048))                    # 671 MB of populations: HBM-bound, one launch per step
    assert big.stepping == "launch"
    big.close()


# ------------------------------------------------------------------------------------------- prescribed fields
@pytest.mark.parametrize("pattern", ["pull2", "aa"])
@pytest.mark.parametrize("precision,n,ny,steps", [("f64", 48, 31, 120), ("f64s", 40, 40, 60), ("f32s", 64, 37, 200)])
def test_swe_over_a_bed_matches_the_oracle(P, precision, n, ny, steps, pattern):
    """eq (3.5)-(3.6): S = -g h grad z_b with the bed slope as a prescribed per-node field, SM5.3 fields
    (L1200-L1207) with forcing on."""
    w = W.relabel(W.pin_swe(n, precision=precision), ny=ny)
    U, f, _ = gpu_run(P, w, steps, pattern=pattern, stepping="launch")
    Uo, fo = oracle_run(w, steps)
    tol = {"f64": 1e-12, "f64s": 1e-11, "f32s": 2e-5}[precision]
    gate(U, Uo, fo, precision, f"{w.name}[{pattern}]", U_ref=w.U_ref, tol=tol, steps=steps)
    if precision == "f64":
        assert np.abs(f - fo).max() / np.abs(fo).max() <= 1e-12


def test_bed_source_is_what_changes_the_flow(P):
    """The prescribed field is really read: zero slope gives the flat-bottom system (to rounding: the two specialisations are
    compiled separately), a non-zero slope does not."""
    w = W.pin_swe(32)
    flat = W.relabel(w, system="swe2d", params=w.params, mms_id=0, mms_params=[], aux=None)
    wb = W.relabel(w, mms_id=0)
    g0 = P.Grid.from_workload(flat, pattern="pull2"); g0.init_from_U(w.initial_U()); g0.step(20); f0 = g0.read_populations(); g0.close()
    for scale, same in ((0.0, True), (1.0, False)):
        g = P.Grid.from_workload(wb, pattern="pull2")
        g.set_aux_fields(scale * wb.aux_fields())
        g.init_from_U(w.initial_U()); g.step(20)
        f = g.read_populations(); g.close()
        d = np.abs(f - f0).max() / np.abs(f0).max()
        assert (d <= 1e-13) if same else (d > 1e-7), d


@pytest.mark.parametrize("pattern", ["pull2", "aa"])
@pytest.mark.parametrize("precision,shape,steps", [("f64", (20, 12, 9), 40), ("f32s", (32, 10, 12), 60)])
def test_hcnsf_matches_the_oracle_with_time_dependent_prescribed_fields(P, precision, shape, steps, pattern):
    """eq (3.27): porosity alpha(x,t) and solid velocity u_s(x,t) are per-node inputs, refreshed before
    every step at t_n + dt/2 (L154) on both sides from the same workload recipe (SM5.13-SM5.14, L1424-L1434)."""
    n, ny, nz = shape
    w = W.hcnsf3d(n, ny=ny, nz=nz, precision=precision)
    g = P.Grid.from_workload(w, pattern=pattern)
    g.init_from_U(w.initial_U())
    for s in range(steps):
        g.set_aux_fields(w.aux_fields((s + 0.5) * w.dt))
        g.step(1)
    U = g.read_U()
    speeds, status = g.max_wave_speed()
    g.close()
    Uo, fo = oracle_run(w, steps, aux_in_time=True)
    gate(U, Uo, fo, precision, f"{w.name}[{pattern}]", U_ref=w.U_ref, steps=steps)
    assert status == 0 and 0.05 < max(speeds[:2]) < 0.5


def test_prescribed_field_calls_are_refused_out_of_order(P):
    w = W.pin_swe(16)
    s = P.System(w.system, params=w.params, tau_R=w.tau_R)
    g = P.Grid(s, 16, 16, 1, w.dx, w.lam)
    with pytest.raises(P.LbmkError) as e:                     # init before the prescribed fields are set
        g.init_from_U(w.initial_U())
    assert e.value.status == 5
    g.close()
    e2 = P.Grid.from_workload(W.c3_euler(16))
    with pytest.raises(P.LbmkError) as e:                     # a system without prescribed fields
        P.lbmk_set_aux_fields(e2.h, e2.workspace.data_ptr(), True)
    assert e.value.status == 6
    e2.close()


# ------------------------------------------------------------------------------------------- resistive MHD 2D
@pytest.mark.parametrize("pattern", ["pull2", "aa"])
@pytest.mark.parametrize("precision,n,ny,steps", [("f64", 40, 27, 200), ("f64s", 32, 32, 100), ("f32s", 128, 20, 400)])
def test_mhd2d_matches_the_oracle(P, precision, n, ny, steps, pattern):
    """eq (3.25): 6 conserved + 12 tracker fields, viscous stress / heat flux / resistive terms by the chain
    rule, Powell source from tr G_B; SM5.12 fields (L1375-L1392) with forcing on; moving, magnetised reference state."""
    w = W.relabel(W.pin_mhd2d(n, precision=precision), ny=ny)
    U, f, _ = gpu_run(P, w, steps, pattern=pattern)
    Uo, fo = oracle_run(w, steps)
    tol = {"f64": 1e-12, "f64s": 1e-11, "f32s": 2e-5}[precision]
    # fp32: the six conserved fields are gated strictly; the lattice-unit trackers G = dx grad V are O(dx) quantities fed by
    # their O(1..10) parents (Mach-3, magnetised reference) through -V/g_tau, so their rounding is the parents' (eps32 |V|),
    # not their own: cancellation-scaled rule of tests/parity_metric.py, each figure recorded in the parity table
    strict = True if precision != "f32s" else [True] * 6 + [False] * 12
    gate(U, Uo, fo, precision, f"{w.name}[{pattern}]", U_ref=w.U_ref, tol=tol, steps=steps, strict=strict)


def test_mhd2d_subcharacteristic_reduction_matches_the_oracle(P):
    w = W.pin_mhd2d(48)
    g = P.Grid.from_workload(w); g.init_from_U(w.initial_U()); g.step(30)
    sp, status = g.max_wave_speed(); g.close()
    o = oracle.OracleGrid.from_workload(w); o.init_from_U(w.initial_U()); o.step(30)
    so = o.max_wave_speed(); o.close()
    assert status == 0 and np.allclose(sp, so, rtol=1e-11)


# ------------------------------------------------------------------------------------------- generated vs hand-written flux
@pytest.mark.parametrize("mk,kw,prec,steps", [
    (W.pin_euler, dict(n=48), "f64s", 40), (W.pin_swe, dict(n=40), "f64", 30), (W.pin_adr, dict(n=32), "f64s", 60),
    (W.pin_allencahn, dict(n=32), "f64", 60), (W.pin_inse, dict(n=32), "f64s", 60), (W.pin_nsf2d, dict(n=40), "f64s", 80),
    (W.pin_mhd2d, dict(n=40), "f64s", 80), (W.c4_nsf3d, dict(n=16, ny=12, nz=10), "f64s", 30), (W.c4_nsf3d, dict(n=16, ny=12, nz=10), "f32s", 30),
    (W.c1_advection, dict(n=40, ny=24), "f64", 10), (W.pin_burgers, dict(n=32), "f64", 30), (W.c2_swe, dict(n=40, ny=28), "f64s", 30),
    (W.pin_urf, dict(n=32), "f64", 30), (W.pin_maxwell, dict(n=32), "f64", 30), (W.pin_elasticity, dict(n=32), "f64s", 30),
    (W.hcnsf3d, dict(n=16, ny=12, nz=10), "f64s", 20), (W.hcnsf3d, dict(n=16, ny=12, nz=10), "f32s", 20),
    (W.c5_mhd3d, dict(n=16, ny=12, nz=10), "f64s", 20), (W.c5_mhd3d, dict(n=16, ny=12, nz=10), "f32s", 20)])
def test_hand_written_delta_forms_equal_the_generated_augmented_systems(P, mk, kw, prec, steps):
    """gen/cascade.py DERIVES the augmented system (Alg 2.1 Split/Cascade/Assemble/Emit);
    lbmk_flux_selfcheck evaluates, on every node of a live state, the hand-written delta-form flux/source the step kernels use and
    the emitted plain form, both in fp64: they agree to rounding (reference state subtracted analytically vs numerically)."""
    w = mk(**kw)
    g = P.Grid.from_workload(w, precision=prec)
    g.init_from_U(w.initial_U())
    g.step(steps)
    d = P.lbmk_flux_selfcheck(g.h)
    g.close()
    assert 0.0 <= d <= 5e-12, d


def test_every_system_has_a_generated_form(P):
    """All 16 systems of the library carry the emitted plain form next to their hand-written delta form."""
    for name in P.SYSTEM_ID:
        mk = {"advection2d": W.c1_advection, "burgers2d": W.pin_burgers, "swe2d": W.c2_swe, "euler2d": W.pin_euler, "adr2d": W.pin_adr,
              "nsf3d": W.c4_nsf3d, "mhd3d": W.c5_mhd3d, "urf2d": W.pin_urf, "maxwell2d": W.pin_maxwell, "allencahn2d": W.pin_allencahn,
              "inse2d": W.pin_inse, "elasticity2d": W.pin_elasticity, "nsf2d": W.pin_nsf2d, "swe2d_bathy": W.pin_swe,
              "hcnsf3d": W.hcnsf3d, "mhd2d": W.pin_mhd2d}[name]
        w = mk(n=16 if name in ("nsf3d", "mhd3d", "hcnsf3d") else 32)
        assert w.system == name
        g = P.Grid.from_workload(w); g.init_from_U(w.initial_U()); g.step(3)
        d = P.lbmk_flux_selfcheck(g.h)
        g.close()
        assert 0.0 <= d <= (5e-12 if w.precision == "f64" else 5e-5), (name, d)


def test_multi_node_kernel_for_single_field_fp32_is_bit_identical(P):
    """Single-field fp32 systems on grids of >= 128*4*SMs nodes step with 4 nodes per thread (collide_stream_multi): same bits as the
    one-node-per-thread code (the persistent kernel runs node_step), same parity against the oracle; ragged tail, odd sizes."""
    w = W.relabel(W.pin_burgers(301, precision="f32s"), ny=277, mms_id=0)          # 83 377 nodes, not a multiple of anything
    U1, f1, (m1, l1) = gpu_run(P, w, 9, [1, 8], pattern="pull2", stepping="launch")
    U2, f2, (m2, l2) = gpu_run(P, w, 9, [1, 8], pattern="pull2", stepping="persistent")
    assert (m1, m2) == ("launch", "persistent") and np.array_equal(f1, f2)
    Uo, fo = oracle_run(w, 9)
    gate(U1, Uo, fo, "f32s", f"{w.name}[multi]", U_ref=w.U_ref, steps=9, strict=False)


def test_host_U_moves_in_chunks_and_equals_the_device_path(P):
    """lbmk_init_from_U / lbmk_read_U with HOST buffers go through two fixed staging buffers in node chunks (4 chunks here, the last
    one ragged; pageable and pinned memory): same populations and same U as with device buffers."""
    import torch
    w = W.c4_nsf3d(n=96, ny=96, nz=97, mms=False)                    # 893 952 nodes x 17 fields: 121 MB of fp64 U, chunks of 246 656 nodes
    U0 = w.initial_U()
    g = P.Grid.from_workload(w); g.init_from_U(torch.from_numpy(U0).cuda()); g.step(3)
    f_dev = g.read_populations(); U_dev = g.read_U(torch.empty(U0.shape, dtype=torch.float64, device="cuda")).cpu().numpy()
    g.close()
    for pinned in (False, True):
        src = torch.from_numpy(U0).pin_memory() if pinned else torch.from_numpy(U0)
        g = P.Grid.from_workload(w); g.init_from_U(src); g.step(3)
        assert np.array_equal(g.read_populations(), f_dev)
        out = torch.empty(U0.shape, dtype=torch.float64, pin_memory=pinned)
        U_host = g.read_U(out)
        g.close()
        assert np.array_equal(np.asarray(U_host), U_dev)


@pytest.mark.parametrize("mk,kw,steps", [
    (W.c5_mhd3d, dict(n=40, ny=36, nz=30), 9),                       # 3D: 338 tiles, stencil reach nx*ny = 11.25 tiles -> dependency runs of ~24 blocks, cyclic wrap in z
    (lambda **kw: W.relabel(W.c2_swe(**kw), mms_id=0), dict(n=512, ny=301), 11),   # 1204 tiles: several tiles per block, last block short
    (W.c3_euler, dict(n=130, ny=517), 10),                           # rows straddle tiles and blocks, ragged last tile
    (W.c2_swe, dict(n=512, ny=300), 13),                             # forcing on, >= 8 segments per SM: FAT persistent blocks (boundary segments first)
    (W.c2_swe, dict(n=64, ny=2401), 12),                             # narrow rows: reach = half a segment, nearly all segments interior; ragged
    (W.c3_euler, dict(n=1000, ny=160), 8),                           # fp32, reach = 7.8 segments of the 9 a block owns: no interior
])
def test_step_flags_between_neighbouring_blocks_many_blocks(P, mk, kw, steps):
    """The launch-free kernels synchronise neighbouring blocks with point-to-point step flags (kernels.cuh dependency_run): grids with
    hundreds of co-resident blocks, partial dependency runs, cyclic wrap and a short last block give the per-launch bits -- persistent
    (thin 128-thread blocks, and from 8 segments per SM on the fat 512-thread blocks that publish their flag after the boundary
    segments and hide its round trip behind the interior ones) against two-lattice per-launch, SM-resident against AA per-launch."""
    w = mk(**kw)
    U1, f1, (m1, _) = gpu_run(P, w, steps, [1, steps - 1], pattern="pull2", stepping="launch")
    U2, f2, (m2, _) = gpu_run(P, w, steps, [1, steps - 1], pattern="pull2", stepping="persistent")
    assert (m1, m2) == ("launch", "persistent") and np.array_equal(f1, f2)
    U3, f3, (m3, _) = gpu_run(P, w, steps, [1, steps - 1], pattern="aa", stepping="launch")
    U4, f4, (m4, _) = gpu_run(P, w, steps, [1, steps - 1], stepping="resident")
    assert (m3, m4) == ("launch", "resident") and np.array_equal(f3, f4)
    d = np.abs(f3 - f1).max() / np.abs(f1).max()
    assert d <= (2e-6 if w.precision == "f32s" else 1e-13), d        # AA and two-lattice kernels: same arithmetic, separately compiled
