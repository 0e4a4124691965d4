"""lbmk_error_norms_noalloc (include/lbmk.h): the error norms for callers that must not allocate -- the scratch of its two-pass
reduction is a static device array inside the library, found with cudaGetSymbolAddress once per device.

Collected last on purpose (the suite runs with pytest -x): checks the entry point against the existing lbmk_error_norms on two
calls in a row that SHARE the static scratch -- a large grid first, a small one second, so stale records of the first call sit
behind the records of the second -- plus a repeat (bit-reproducible), the size limit and the state checks.  Passes alone in a
fresh process and after the rest of the suite."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
TOL64 = 1e-12     # BASELINE.json north_star: fp64 tolerance of the parity tests


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2607_05668_b200 as P
    P.lib()
    return P


def _both(P, g, out):
    """(existing path, new entry point) on the grid's current state; `out` is a preallocated device tensor."""
    import torch
    ref = P.lbmk_error_norms(g.h, g.system.m_total)
    out.fill_(-1.0)
    P.lbmk_error_norms_noalloc(g.h, out.data_ptr())
    torch.cuda.synchronize()
    return ref, out.cpu().numpy().copy()


def _check(ref, got):
    sums, maxs = [0, 1, 3, 4], [2, 5]
    assert np.isfinite(got).all() and (got >= 0).all()
    assert np.array_equal(got[:, maxs], ref[:, maxs])                                  # maxima: exact
    assert np.abs(got[:, sums] - ref[:, sums]).max() <= TOL64 * np.abs(ref[:, sums]).max()
    rel = np.abs(got[:, sums] - ref[:, sums]) / np.maximum(np.abs(ref[:, sums]), 1e-300)
    assert rel.max() <= 1e-10                                                          # each sum of ~1e6 terms on its own scale


def test_no_alloc_error_norms_match_the_existing_path_on_two_calls_in_a_row(P):
    import torch
    big = W.c4_nsf3d(n=96, ny=80, nz=70)                  # 537 600 nodes, 17 fields, fp32 shifted: 132 records (the last one ragged)
    small = W.c2_swe(n=200, ny=37)                        # 7 400 nodes, 3 fields, fp64: 2 records
    out_big = torch.empty((17, 6), dtype=torch.float64, device="cuda")
    out_small = torch.empty((3, 6), dtype=torch.float64, device="cuda")
    gb = P.Grid.from_workload(big); gb.init_from_U(big.initial_U()); gb.step(6)
    gs = P.Grid.from_workload(small); gs.init_from_U(small.initial_U()); gs.step(9)
    ref_b, got_b = _both(P, gb, out_big)                  # call 1
    ref_s, got_s = _both(P, gs, out_small)                # call 2: same scratch, stale records of call 1 behind its own
    _check(ref_b, got_b)
    _check(ref_s, got_s)
    assert (got_s[:, 1] > 0).all() and (got_b[:, 4] > 0).all()       # real, non-trivial sums (the non-square grid is not a convergence case)
    # fixed reduction tree: a repeat gives the same bits; AA storage at an odd step count goes through the same gather
    _, again = _both(P, gs, out_small)
    assert np.array_equal(again, got_s)
    gs.step(1)
    _check(*_both(P, gs, out_small))
    gs.close(); gb.close()
    ga = P.Grid.from_workload(small, pattern="aa"); ga.init_from_U(small.initial_U()); ga.step(9)
    ref_a, got_a = _both(P, ga, out_small)
    _check(ref_a, got_a)
    ga.close()


def test_no_alloc_error_norms_bounded_grid(P):
    """Dirichlet-MMS frame: the frame refresh before the reduction is part of the entry point, as in lbmk_error_norms."""
    import torch
    w = W.pin_euler(n=40)
    out = torch.empty((4, 6), dtype=torch.float64, device="cuda")
    g = P.Grid.from_workload(w, bc="dirichlet_mms"); g.init_from_U(w.initial_U()); g.step(12)
    _check(*_both(P, g, out))
    g.close()


def test_no_alloc_error_norms_limits_and_misuse(P):
    import torch
    # beyond the static scratch: 4608^2 nodes x 18 fields need 5184 records x 864 B = 4.48 MB > 4 MiB.  Refused from the grid's size
    # alone, before any workspace exists (so the test allocates nothing)
    w = W.pin_mhd2d(n=64)
    s = P.System(w.system, params=w.params, tau_R=w.tau_R, g_tau=w.g_tau, U_ref=w.U_ref, mms_id=w.mms_id, mms_params=w.mms_params)
    dummy = torch.empty((18, 6), dtype=torch.float64, device="cuda")
    n = 4608
    g = P.lbmk_grid_create(s.h, n, n, 1, 0, 1.0 / n, w.lam, P.LBMK_F32_SHIFTED, torch.cuda.current_stream().cuda_stream)
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_error_norms_noalloc(g, dummy.data_ptr())
    assert e.value.status == 1 and "static scratch" in str(e.value) and str(P.LBMK_NOALLOC_SCRATCH_BYTES) in str(e.value)
    P.lbmk_grid_destroy(g)
    # the largest square MHD 2D grid that fits (4854 records): accepted as far as its size goes, then refused for its state
    n = 4456
    assert -(-n * n // 4096) * 18 * 48 <= P.LBMK_NOALLOC_SCRATCH_BYTES
    g = P.lbmk_grid_create(s.h, n, n, 1, 0, 1.0 / n, w.lam, P.LBMK_F32_SHIFTED, torch.cuda.current_stream().cuda_stream)
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_error_norms_noalloc(g, dummy.data_ptr())
    assert e.value.status == 5                                   # LBMK_ESTATE: no workspace bound
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_error_norms_noalloc(g, 0)
    assert e.value.status == 1
    P.lbmk_grid_destroy(g)
    s.close()
    # no manufactured solution: unsupported, as for lbmk_error_norms
    w0 = W.c1_advection()
    g0 = P.Grid.from_workload(w0); g0.init_from_U(w0.initial_U())
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_error_norms_noalloc(g0.h, dummy.data_ptr())
    assert e.value.status == 6
    g0.close()
