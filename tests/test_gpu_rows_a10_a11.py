"""GPU parity of SURVEY.md §8(a) rows a10 (sub-characteristic check) and a11 (Dirichlet-MMS frame), and
element-by-element parity on grids whose x extent is a multiple of the thread-block size, where the step
kernel takes its forcing coefficients from the shared-memory copy of the row (csrc/kernels.cuh `staged`)."""
import numpy as np
import pytest

import oracle
import workloads as W
from parity_metric import gate

pytestmark = pytest.mark.gpu
TOL64, TOL32 = 1e-12, 2e-5     # BASELINE.json north_star


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2607_05668_b200 as P
    P.lib()
    return P


def _pair(P, w, steps, bc="periodic", **kw):
    U0 = w.initial_U()
    g = P.Grid.from_workload(w, bc=bc, **kw)
    g.init_from_U(U0)
    g.step(steps)
    U = g.read_U()
    ws = g.max_wave_speed()
    g.close()
    o = oracle.OracleGrid.from_workload(w, bc=bc)
    o.init_from_U(U0)
    o.step(steps)
    Uo, fo, wo = o.read_U(), o.read_f(), o.max_wave_speed()
    o.close()
    return U, Uo, fo, ws, wo


# ---------------------------------------------------------------------------------------------- a10
@pytest.mark.parametrize("name,kw,steps,tol", [
    ("c1", dict(n=40, ny=24), 5, 1e-13), ("c2", dict(n=48, ny=20), 7, 1e-12),
    ("c3", dict(n=64, ny=24), 9, 1e-5), ("c4", dict(n=16, ny=12, nz=10), 6, 1e-5), ("c5", dict(n=16, ny=12, nz=10), 6, 1e-5)])
@pytest.mark.parametrize("pattern", ["pull2", "aa"])
def test_a10_device_wave_speed_reduction_matches_oracle(P, name, kw, steps, tol, pattern):
    """eq (2.19)-(2.20): per-axis, isotropic and tracker-coupling lattice speeds after an odd and
    an even number of steps (the reduction gathers the canonical state from either storage pattern)."""
    w = W.BASELINE_CONFIGS[name](**kw)
    for st in (steps, steps + 1):
        U, Uo, fo, (speeds, status), wo = _pair(P, w, st, pattern=pattern)
        assert status == 0
        for a, b in zip(speeds, wo):
            assert a == pytest.approx(b, rel=tol, abs=1e-15)
        cs = np.sqrt(1.0 / 3.0 if w.dim == 2 else 0.25)
        assert max(speeds[0], speeds[1]) + speeds[2] <= cs


def test_a10_violation_is_reported(P):
    """Lattice wave speed above c_s: refused a priori at grid creation when the bound is declared (LBMK_ESUBCHAR),
    detected by the device reduction when it is not."""
    w = W.relabel(W.c3_euler(n=32), lam=1.2)            # sound speed 1 => lattice speed 0.83 > c_s = 0.577
    with pytest.raises(P.LbmkError) as e:
        P.Grid.from_workload(w)
    assert e.value.status == 4
    g = P.Grid.from_workload(w, declare_bound=False)
    g.init_from_U(w.initial_U())
    speeds, status = g.max_wave_speed()
    assert status == 4 and speeds[1] > np.sqrt(1.0 / 3.0)
    with pytest.raises(P.LbmkError):
        g.check_subcharacteristic()
    g.close()


def test_a10_blown_up_state_is_reported(P):
    """A state that has ALREADY blown up (NaN after a sub-characteristic violation) must not pass
    the device check: fmax() drops NaN operands, so the reduction maps non-finite wave speeds to +inf explicitly."""
    w = W.relabel(W.c3_euler(n=32, precision="f64"), lam=1.2)
    g = P.Grid.from_workload(w, declare_bound=False)
    g.init_from_U(w.initial_U())
    for _ in range(40):
        g.step(50)
        if not np.isfinite(g.read_U()).all():
            break
    assert not np.isfinite(g.read_U()).all(), "the lam = 1.2 Euler run was expected to blow up"
    speeds, status = g.max_wave_speed()
    assert status == 4 and not (max(speeds[0], speeds[1]) <= np.sqrt(1.0 / 3.0))
    g.close()
    # every node NaN
    g = P.Grid.from_workload(W.c3_euler(n=16, precision="f64"))
    g.init_from_U(np.full(g.shape_U, np.nan))
    speeds, status = g.max_wave_speed()
    assert status == 4 and np.isinf(speeds[0])
    g.close()


# ---------------------------------------------------------------------------------------------- a11
@pytest.mark.parametrize("mk,kw,steps,tol", [
    (W.c2_swe, dict(n=40, ny=28), 33, TOL64), (W.pin_burgers, dict(n=24), 40, TOL64), (W.pin_euler, dict(n=20), 30, TOL64),
    (W.c4_nsf3d, dict(n=12, ny=10, nz=9, precision="f64"), 14, TOL64), (W.c4_nsf3d, dict(n=14, ny=10, nz=9), 20, TOL32)])
def test_a11_dirichlet_mms_frame_parity(P, mk, kw, steps, tol):
    """Reading A18: the outermost node layer is reset to f_eq(Q_exact(x_b, t_n)) before every step and before
    readback; the interior is the ordinary step.  Same construction on both sides, compared element by element."""
    w = mk(**kw)
    U, Uo, fo, _, _ = _pair(P, w, steps, bc="dirichlet_mms")
    gate(U, Uo, fo, w.precision, f"{w.name}[dirichlet]", U_ref=w.U_ref, tol=tol, steps=steps)
    # the frame holds the exact state at the final time
    o = oracle.OracleGrid.from_workload(w, bc="dirichlet_mms")
    Ue = o.exact_U(steps * w.dt)
    o.close()
    frame = np.ones(U.shape[1:], dtype=bool)
    inner = (slice(1, -1) if w.dim == 3 else slice(None), slice(1, -1), slice(1, -1))
    frame[inner] = False
    scale = np.abs(Ue).reshape(U.shape[0], -1).max(axis=1).reshape(-1, 1) + 1e-300
    assert (np.abs(U - Ue)[:, frame] / scale).max() <= (1e-12 if tol == TOL64 else 1e-5)


# ------------------------------------------------------------------------ staged forcing coefficients
@pytest.mark.parametrize("mk,kw,steps,tol", [
    (W.c4_nsf3d, dict(n=128, ny=6, nz=5), 12, TOL32),                       # nx = 2 blocks of 64 (c4 fp32 launch shape): staged, fp32 shifted
    (W.c4_nsf3d, dict(n=256, ny=4, nz=3, precision="f64"), 6, TOL64),
    (W.c2_swe, dict(n=256, ny=12), 40, TOL64),                              # nx = 2 blocks of 128 (2D launch shape): staged, fp64
    (W.c2_swe, dict(n=512, ny=9, precision="f32s"), 40, TOL32),
    (W.pin_burgers, dict(n=256), 20, TOL64)])
@pytest.mark.parametrize("pattern", ["pull2", "aa"])
def test_staged_row_coefficients_parity(P, mk, kw, steps, tol, pattern):
    w = mk(**kw)
    U, Uo, fo, _, _ = _pair(P, w, steps, pattern=pattern)
    gate(U, Uo, fo, w.precision, f"{w.name}[staged,{pattern}]", U_ref=w.U_ref, tol=tol, steps=steps, strict=False)   # short runs
    # many short lbmk_step calls (coefficient batches restart at every call) give the same state as one long call
    g = P.Grid.from_workload(w, pattern=pattern)
    g.init_from_U(w.initial_U())
    for _ in range(steps):
        g.step(1)
    U1 = g.read_U()
    g.close()
    assert np.array_equal(U1, U)


# ------------------------------------------------------------------------ degenerate grids
@pytest.mark.parametrize("name,kw", [("c3", dict(n=1, ny=1, precision="f64")), ("c3", dict(n=1, ny=9, precision="f64")),
                                     ("c3", dict(n=7, ny=1)), ("c5", dict(n=1, ny=1, nz=1, precision="f64")),
                                     ("c5", dict(n=1, ny=3, nz=2)), ("c4", dict(n=2, ny=1, nz=1, precision="f64")),
                                     ("c1", dict(n=1, ny=2))])
@pytest.mark.parametrize("pattern", ["pull2", "aa"])
def test_degenerate_grids_parity(P, name, kw, pattern):
    """One-node axes: every neighbour along such an axis is the node itself (periodic wrap onto itself)."""
    w = W.BASELINE_CONFIGS[name](**kw)
    U, Uo, fo, _, _ = _pair(P, w, 7, pattern=pattern)
    gate(U, Uo, fo, w.precision, f"{w.name}[degenerate,{pattern}]", U_ref=w.U_ref, steps=7, strict=False)   # vanishing fields


# ------------------------------------------------------------------------ out-of-bounds guard (no sanitizer on this pool)
@pytest.mark.parametrize("mk,kw", [(W.c1_advection, dict(n=37, ny=23)), (W.c4_nsf3d, dict(n=5, ny=4, nz=3)), (W.c4_nsf3d, dict(n=130, ny=3, nz=2)),
                                   (W.c5_mhd3d, dict(n=9, ny=2, nz=5)), (W.c2_swe, dict(n=257, ny=3)), (W.pin_nsf2d, dict(n=19)),
                                   (W.pin_swe, dict(n=21)), (W.hcnsf3d, dict(n=7, ny=5, nz=3)), (W.pin_mhd2d, dict(n=13))])
@pytest.mark.parametrize("pattern,stepping", [("pull2", "launch"), ("aa", "launch"), ("pull2", "persistent"), ("pull2", "cluster"), ("aa", "resident")])
def test_workspace_guards_stay_untouched(P, mk, kw, pattern, stepping):
    """The workspace is bound inside a larger buffer filled with a sentinel; after init, steps (ragged last tile, wraps
    on every axis, forcing tables, prescribed fields; per-launch, persistent, cluster-resident and SM-resident stepping), reductions,
    readbacks and the flux self-check the guard bands before and after it are unchanged (compute-sanitizer is closed on this pool)."""
    import torch
    w = mk(**kw)
    s = P.System(w.system, params=w.params, tau_R=w.tau_R, g_tau=w.g_tau, U_ref=w.U_ref, mms_id=w.mms_id,
                 mms_params=w.mms_params if w.mms_id else ())
    prec = {"f64": P.LBMK_F64, "f32s": P.LBMK_F32_SHIFTED}[w.precision]
    g = P.lbmk_grid_create(s.h, w.nx, w.ny, w.nz, 0, w.dx, w.lam, prec, torch.cuda.current_stream().cuda_stream)
    P.lbmk_grid_set_option(g, P.LBMK_OPT_PATTERN, P.PATTERN[pattern])
    P.lbmk_grid_set_option(g, P.LBMK_OPT_STEPPING, P.STEPPING[stepping])
    nbytes = P.lbmk_grid_workspace_bytes(g)
    G = 1 << 16
    buf = torch.full((nbytes + 2 * G + 256,), 0xA5, dtype=torch.uint8, device="cuda")
    off = (-buf.data_ptr()) % 256 + G
    P.lbmk_grid_bind_workspace(g, buf.data_ptr() + off, nbytes)
    U0 = torch.from_numpy(w.initial_U()).cuda()
    out = torch.empty_like(U0)
    if w.n_aux:
        A = torch.from_numpy(w.aux_fields()).cuda()
        P.lbmk_set_aux_fields(g, A.data_ptr(), True)
    P.lbmk_init_from_U(g, U0.data_ptr(), True)
    for n in (1, 2, 5):
        P.lbmk_step(g, n)
        P.lbmk_read_U(g, out.data_ptr(), True)
        P.lbmk_check_subcharacteristic(g, raise_on_violation=False)
    P.lbmk_flux_selfcheck(g)
    torch.cuda.synchronize()
    assert bool((buf[:off] == 0xA5).all()) and bool((buf[off + nbytes:] == 0xA5).all())
    assert bool(torch.isfinite(out).all())
    P.lbmk_grid_destroy(g)
    s.close()
