"""Convergence study on the device: `lbmk_error_norms` against NumPy norms, and the paper's
Table 2 rows (double precision, N = 512, t = 1) reproduced by the CUDA path itself."""
import math

import numpy as np
import pytest

import oracle
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


@pytest.mark.parametrize("mk,kw,steps", [
    (W.pin_burgers, dict(n=40), 30), (W.pin_euler, dict(n=36), 25), (W.pin_adr, dict(n=32), 40), (W.c2_swe, dict(n=48, ny=20), 21),
    (W.c4_nsf3d, dict(n=16, ny=12, nz=10, precision="f64"), 9), (W.c4_nsf3d, dict(n=16, ny=12, nz=10), 8),
    (W.pin_urf, dict(n=32), 17), (W.pin_maxwell, dict(n=32), 16), (W.pin_allencahn, dict(n=32), 40), (W.pin_inse, dict(n=32), 40), (W.pin_elasticity, dict(n=32), 40), (W.pin_nsf2d, dict(n=32), 40),
    (W.pin_swe, dict(n=40), 33), (W.pin_mhd2d, dict(n=32), 40)])
@pytest.mark.parametrize("pattern", ["pull2", "aa"])
def test_error_norms_match_numpy(P, mk, kw, steps, pattern):
    """Device reductions vs norms formed in NumPy from the read-back state and the ORACLE's exact fields (jets)."""
    w = mk(**kw)
    g = P.Grid.from_workload(w, pattern=pattern)
    g.init_from_U(w.initial_U())
    g.step(steps)
    U = g.read_U()
    got = g.error_norms()
    g.close()
    o = oracle.OracleGrid.from_workload(w)
    Ue = o.exact_U(steps * w.dt)
    o.close()
    for k in range(w.m_total):
        e, q = np.abs(U[k] - Ue[k]), np.abs(Ue[k])
        want = (e.sum() / q.sum(), math.sqrt((e * e).sum() / (q * q).sum()), e.max() / q.max())
        for a, b in zip(got[k], want):
            assert a == pytest.approx(b, rel=1e-8, abs=1e-18), (w.name, k, got[k], want)


def test_error_norms_need_a_manufactured_solution(P):
    w = W.c3_euler(n=32)
    g = P.Grid.from_workload(w)
    g.init_from_U(w.initial_U())
    with pytest.raises(P.LbmkError) as e:
        g.error_norms()
    assert e.value.status == 6
    g.close()


def _sig5(a, b):
    return abs(a - b) <= 1.01e-4 * abs(b)


# printed in PAPER.md Table 2 (Double, N = 512): field -> (rel Linf, rel L2); vector fields = root-sum-square (A7)
TABLE2 = [
    (W.pin_burgers, {"u": ((0,), 6.1175e-04, 8.5671e-05)}, "L518"),
    (W.pin_euler, {"rho": ((0,), 1.4401e-06, 6.8435e-07), "E": ((3,), 3.3385e-06, 1.8316e-06), "rhou": ((1, 2), 3.2141e-06, 1.8745e-06)}, "L519-L522"),
    (W.pin_urf, {"E": ((0,), 4.3449e-06, 2.1354e-06), "S": ((1, 2), 9.6256e-06, 6.3943e-06)}, "L527-L529"),
    (W.pin_maxwell, {"Ez": ((0,), 2.9956e-05, 2.9956e-05), "Hx": ((1,), 1.0951e-04, 1.0951e-04), "Hy": ((2,), 1.1587e-05, 1.1587e-05)}, "L530-L535"),
    (W.pin_adr, {"c": ((0,), 2.2901e-04, 1.2680e-04)}, "L540"),
    (W.pin_allencahn, {"phi": ((0,), 7.3196e-04, 7.8653e-04)}, "L542"),
    (W.pin_elasticity, {"F": ((0, 1, 2, 3), 3.1874e-05, 2.8940e-05), "v": ((4, 5), 6.4804e-05, 4.5664e-05)}, "L536-L539"),
    (W.pin_swe, {"h": ((0,), 5.5560e-06, 2.3433e-06), "hu": ((1, 2), 2.6837e-05, 2.0838e-05)}, "L523-L526"),   # c2's own system, with the bed
    # the paper's running example: 4 conserved fields + 8 chain-rule trackers, 131 072 steps; mu = K = 0.01 (reading A24)
    (W.pin_nsf2d, {"rho": ((0,), 7.3384e-05, 3.7592e-05), "rhou": ((1, 2), 1.1775e-04, 6.8579e-05), "E": ((3,), 8.3354e-05, 4.5785e-05)}, "L547-L551"),
]


@pytest.mark.parametrize("mk,fields,cite", TABLE2)
def test_paper_table2_double_rows_reproduced_on_the_gpu(P, mk, fields, cite):
    """The whole study of one Table 2 row on the device: N = 512, fp64, round(1/dt) steps with manufactured forcing,
    relative errors at the final time -- equal to the printed values to their 5 significant digits."""
    w = mk(512)
    g = P.Grid.from_workload(w)
    g.init_from_U(w.initial_U())
    g.step(w.steps)
    n = g.error_norms()
    g.close()
    for name, (ks, linf, l2) in fields.items():
        got_linf = math.sqrt(sum(n[k][2] ** 2 for k in ks))
        got_l2 = math.sqrt(sum(n[k][1] ** 2 for k in ks))
        print(f"{w.name} {name}: Linf {got_linf:.4e} (paper {linf:.4e})  L2 {got_l2:.4e} (paper {l2:.4e})  PAPER.md:{cite}")
        assert _sig5(got_l2, l2) and _sig5(got_linf, linf), (w.name, name, got_linf, got_l2)


def test_paper_table2_inse_row_partially_reproduced(P):
    """Weakly compressible NSE.  The listing of its tracker fluxes is inconsistent with eq (3.22)
    (SM4.9 L955: Phi_{4,1}, Phi_{6,1} print rho u_0 where G (x) u gives rho u_1); the vector form is used.  It
    reproduces the printed momentum L2 error to 3 digits; rho (an O(Ma^2) quantity, 6e-7) and the momentum Linf do
    not match to the printed precision -- an unresolved reading, so this system's parity is UNPINNED beyond
    P1/P3/P10/P13.  Gate: momentum L2 within 0.2 %, the rest within 50 %, values printed."""
    w = W.pin_inse(512)
    g = P.Grid.from_workload(w)
    g.init_from_U(w.initial_U())
    g.step(w.steps)
    n = g.error_norms()
    g.close()
    mom_l2, mom_linf = math.hypot(n[1][1], n[2][1]), math.hypot(n[1][2], n[2][2])
    print(f"{w.name}: rho Linf {n[0][2]:.4e} (paper 1.3419e-06) L2 {n[0][1]:.4e} (paper 6.0683e-07); "
          f"rho u Linf {mom_linf:.4e} (paper 8.2447e-04) L2 {mom_l2:.4e} (paper 8.5394e-04)")
    assert abs(mom_l2 - 8.5394e-04) <= 2e-3 * 8.5394e-04
    assert abs(mom_linf - 8.2447e-04) <= 0.5 * 8.2447e-04 and abs(n[0][1] - 6.0683e-07) <= 0.5 * 6.0683e-07


# printed EOCs (Table 2, Double): field -> (components, Linf EOC, L2 EOC); "negative least-squares log-log slope
# over all simulated resolutions" (L514), N = 64, 128, 256, 512 (L499)
TABLE2_EOC = [
    (W.pin_burgers, {"u": ((0,), 1.46, 1.87)}),
    (W.pin_euler, {"rho": ((0,), 1.98, 1.99), "E": ((3,), 2.01, 2.00), "rhou": ((1, 2), 2.00, 2.00)}),
    (W.pin_urf, {"E": ((0,), 2.00, 2.00), "S": ((1, 2), 2.00, 2.00)}),
    (W.pin_maxwell, {"Ez": ((0,), 1.95, 1.95), "Hx": ((1,), 2.00, 2.00), "Hy": ((2,), 2.02, 2.02)}),
    (W.pin_elasticity, {"F": ((0, 1, 2, 3), 2.00, 2.00), "v": ((4, 5), 2.01, 1.99)}),
    (W.pin_adr, {"c": ((0,), 2.50, 2.49)}),
    (W.pin_allencahn, {"phi": ((0,), 2.50, 2.51)}),
    (W.pin_swe, {"h": ((0,), 1.87, 1.88), "hu": ((1, 2), 1.76, 1.70)}),
    (W.pin_nsf2d, {"rho": ((0,), 1.91, 1.95), "rhou": ((1, 2), 1.95, 1.99), "E": ((3,), 1.98, 2.01)}),
]


@pytest.mark.parametrize("mk,fields", TABLE2_EOC)
def test_paper_table2_eoc_reproduced_on_the_gpu(P, mk, fields):
    """The refinement study itself on the device: four resolutions to t = 1 in fp64, LSQ slope of log2(error) vs
    log2(N) -- equal to the printed experimental orders of convergence to their 2 decimals."""
    ns = (64, 128, 256, 512)
    norms = []
    for n in ns:
        w = mk(n)
        g = P.Grid.from_workload(w)
        g.init_from_U(w.initial_U())
        g.step(w.steps)
        norms.append(g.error_norms())
        g.close()
    for name, (ks, eoc_inf, eoc_2) in fields.items():
        for j, want in ((2, eoc_inf), (1, eoc_2)):
            err = [math.sqrt(sum(e[k][j] ** 2 for k in ks)) for e in norms]
            slope = -np.polyfit(np.log2(ns), np.log2(err), 1)[0]
            print(f"{mk.__name__} {name} {'Linf' if j == 2 else 'L2'} EOC {slope:.3f} (paper {want:.2f})")
            assert abs(slope - want) <= 0.0151, (mk.__name__, name, j, slope, want)


def test_fp32_tracks_fp64_over_a_long_diffusive_run(P):
    """ADR to t = 1 at N = 256 (34 493 steps at omega = 1.994) in shifted fp32 against the same run in fp64.  With the
    plainly rounded D2Q5 weights (float(1/3) + 4 float(1/6) = 1 + 3e-8) the zeroth moment drifts linearly in the step
    count (3e-3 at N = 512); with the rest weight taken as 1 - 4 w1 in fp32 (csrc/common.cuh weight0) it does not."""
    res = {}
    for prec in ("f32s", "f64"):
        w = W.pin_adr(256, precision=prec)
        g = P.Grid.from_workload(w)
        g.init_from_U(w.initial_U())
        g.step(w.steps)
        res[prec] = g.read_U()[0]
        g.close()
    d = np.abs(res["f32s"] - res["f64"]).max() / np.abs(res["f64"]).max()
    print(f"ADR N=256, 34493 steps: fp32 vs fp64 max rel diff {d:.3e}")
    assert d < 3e-4


@pytest.mark.parametrize("mk,field,paper_l2", [(W.pin_urf, 0, 4.7227e-06), (W.pin_maxwell, 0, 3.0632e-05)])
def test_paper_table2_float_rows_same_magnitude(P, mk, field, paper_l2):
    """Float rows (same f, tau_R as double for these two systems, Table SM2): rounding differs between
    implementations, so only the magnitude is gated (at most 2x, at least 1/4 of the printed Float value); the value is printed."""
    w = mk(512, precision="f32s")
    g = P.Grid.from_workload(w)
    g.init_from_U(w.initial_U())
    g.step(w.steps)
    l2 = g.error_norms()[field][1]
    g.close()
    print(f"{w.name} shifted fp32: rel L2 {l2:.4e} (paper Float {paper_l2:.4e})")
    assert paper_l2 / 4 <= l2 <= paper_l2 * 2


# ------------------------------------------------------------------------------------------------ fp32 order retained (north_star)
def _l2_by_field(n, fields):
    return {name: math.sqrt(sum(n[k][1] ** 2 for k in ks)) for name, ks in fields.items()}


@pytest.mark.parametrize("mk,fields,paper_float_eoc", [
    (W.pin_euler, {"rho": (0,), "rhou": (1, 2), "E": (3,)}, {"rho": 1.65, "rhou": 1.62, "E": 1.73}),        # PAPER.md:L519-L522 Float rows
    (W.pin_swe, {"h": (0,), "hu": (1, 2)}, {"h": 1.95, "hu": 1.83}),                                         # PAPER.md:L523-L526 Float rows
])
def test_fp32_convergence_order_retained_on_the_config_systems(P, mk, fields, paper_float_eoc):
    """north_star: "<= 2e-5 in shifted fp32, with the fp32 convergence order retained".  The refinement study of the systems of
    configs[2] (Euler) and configs[1] (shallow water, here over the paper's bed) in shifted fp32 at the paper's Float knobs
    (Table SM2) against the SAME study in fp64 at the same knobs: N = 64 ... 512 to t = 1, LSQ L2 slope.  The fp32
    slope stays within 0.5 of the fp64 one (float keeps the order down to a 1e-5 - 1e-4 floor) and within
    0.35 of the Float EOC the paper prints."""
    ns = (64, 128, 256, 512)
    slopes = {}
    for prec in ("f32s", "f64"):
        errs = []
        for n in ns:
            w = mk(n, precision="f32s")                     # Float knobs for both precisions
            g = P.Grid.from_workload(w, precision=prec)
            g.init_from_U(w.initial_U())
            g.step(w.steps)
            errs.append(_l2_by_field(g.error_norms(), fields))
            g.close()
        slopes[prec] = {f: -np.polyfit(np.log2(ns), np.log2([e[f] for e in errs]), 1)[0] for f in fields}
        print(mk.__name__, prec, {f: round(s, 3) for f, s in slopes[prec].items()}, "errors at N=512:", {f: f"{errs[-1][f]:.3e}" for f in fields})
    for f in fields:
        assert abs(slopes["f32s"][f] - slopes["f64"][f]) <= 0.5, (f, slopes)
        assert slopes["f32s"][f] >= 1.2, (f, slopes)
        assert abs(slopes["f32s"][f] - paper_float_eoc[f]) <= 0.35, (f, slopes["f32s"][f], paper_float_eoc[f])


def test_fp32_convergence_order_retained_on_the_running_example(P):
    """Compressible NSF 2D (4 + 8 tracker fields, 131 072 steps at N = 512) in shifted fp32 against the same study in fp64: the L2
    orders stay within 0.15 of the fp64 ones (1.87 / 1.93 / 1.96 against 1.95 / 1.99 / 2.01), the N = 512 errors within 1.5x of the
    fp64 ones and BELOW the Float row the paper prints for its own fp32 run (rho 1.5397e-04, rho u 2.4644e-04,
    E 1.5715e-04 in L2, EOC 1.32 - 1.46)."""
    ns = (64, 128, 256, 512)
    fields = {"rho": (0,), "rhou": (1, 2), "E": (3,)}
    paper_float_l2 = {"rho": 1.5397e-04, "rhou": 2.4644e-04, "E": 1.5715e-04}
    out = {}
    for prec in ("f32s", "f64"):
        errs = []
        for n in ns:
            w = W.pin_nsf2d(n, precision=prec)                 # Table SM2: the same knobs for both precisions
            g = P.Grid.from_workload(w)
            g.init_from_U(w.initial_U())
            g.step(w.steps)
            errs.append(_l2_by_field(g.error_norms(), fields))
            g.close()
        out[prec] = ({f: -np.polyfit(np.log2(ns), np.log2([e[f] for e in errs]), 1)[0] for f in fields}, errs[-1])
        print("pin_nsf2d", prec, {f: round(v, 3) for f, v in out[prec][0].items()}, {f: f"{v:.4e}" for f, v in out[prec][1].items()})
    for f in fields:
        assert abs(out["f32s"][0][f] - out["f64"][0][f]) <= 0.15, (f, out)
        assert out["f64"][1][f] <= out["f32s"][1][f] <= 1.5 * out["f64"][1][f], (f, out)
        assert out["f32s"][1][f] <= paper_float_l2[f], (f, out)


def test_fp32_convergence_order_retained_on_c4(P):
    """configs[3] (NSF 3D + 12 trackers, forcing on) refined N = 32, 64, 128, 256 to the time the config reaches after its 200
    steps at 256^3, in shifted fp32 and in fp64: the L2 slopes of the five conserved fields agree within 0.5 and the fp32
    ones stay above 1.2 (the errors are 1e-5 - 1e-3 here, above the fp32 floor)."""
    ns = (32, 64, 128, 256)
    slopes = {}
    for prec in ("f32s", "f64"):
        errs = []
        for n in ns:
            w = W.c4_nsf3d(n, precision=prec)
            g = P.Grid.from_workload(w)
            g.init_from_U(w.initial_U())
            g.step(200 * n // 256)
            errs.append(g.error_norms()[:5, 1])
            g.close()
        errs = np.array(errs)
        slopes[prec] = [-np.polyfit(np.log2(ns), np.log2(errs[:, k]), 1)[0] for k in range(5)]
        print("c4", prec, np.round(slopes[prec], 3), "L2 errors at 256^3:", errs[-1])
    for k in range(5):
        assert abs(slopes["f32s"][k] - slopes["f64"][k]) <= 0.5 and slopes["f32s"][k] >= 1.2, (k, slopes)


def test_paper_table2_mhd2d_row_within_ten_percent(P):
    """Resistive MHD 2D (knobs L743; fields SM5.12 L1375-L1392).  Built from the vector form (listing SM4.11
    is garbled); the legible listing entries are pinned by P13.  At the printed working point the GPU run is second order and
    lands within 8 % of all eight printed errors (E within 0.7 %), but not on their digits: reading A27, UNPINNED to Table 2
    (a scan of tau_R, g_tau, f and the three diffusivities does not hit all eight at once).  Gate: within 10 %; EOCs of L2
    within 0.15 of the printed ones."""
    paper = {"rho": ((0,), 2.7365e-04, 1.6299e-04, 1.75), "rhou": ((1, 2), 4.6103e-04, 2.4482e-04, 1.88),
             "E": ((3,), 3.6516e-04, 2.1223e-04, 1.96), "B": ((4, 5), 2.4829e-04, 1.6277e-04, 2.22)}
    ns, norms = (64, 128, 256, 512), []
    for n in ns:
        w = W.pin_mhd2d(n)
        g = P.Grid.from_workload(w)
        g.init_from_U(w.initial_U())
        g.step(w.steps)
        norms.append(g.error_norms())
        g.close()
    for name, (ks, linf, l2, eoc) in paper.items():
        got_linf = math.sqrt(sum(norms[-1][k][2] ** 2 for k in ks))
        got_l2 = [math.sqrt(sum(e[k][1] ** 2 for k in ks)) for e in norms]
        slope = -np.polyfit(np.log2(ns), np.log2(got_l2), 1)[0]
        print(f"mhd2d {name}: Linf {got_linf:.4e} (paper {linf:.4e})  L2 {got_l2[-1]:.4e} (paper {l2:.4e})  L2 EOC {slope:.2f} (paper {eoc:.2f})")
        assert abs(got_linf / linf - 1) <= 0.10 and abs(got_l2[-1] / l2 - 1) <= 0.10 and abs(slope - eoc) <= 0.15
