"""Pin P8 / P11: the oracle against the convergence errors the paper PRINTS (Table 2).

tests/golden/paper_pins.json is written by tests/golden/make_paper_pins.py, which calls only `oracle/` and
`workloads/` (never the CUDA path).  It holds, per case, the values printed in the paper (with their citation)
and the oracle's own errors at N = 64 ... 512 from the recipes of SURVEY.md Appendix A (Table SM2 knobs, SM5
exact fields).  Three checks:
  1. the stored N = 512 oracle errors equal the printed ones to the printed precision (5 significant digits);
  2. the oracle AS IT STANDS reproduces the stored N = 64 row (so the stored rows belong to this oracle);
  3. the least-squares convergence order over N = 64 ... 512 lies in the paper's band 1.70-2.51 for L2
      -- P11 on the paper's own cases.
CPU only; the live re-run is N = 64 (seconds).
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
PINS = json.load(open(os.path.join(HERE, "golden", "paper_pins.json")))
MAKERS = {"burgers": W.pin_burgers, "euler": W.pin_euler, "adr": W.pin_adr, "urf": W.pin_urf, "maxwell": W.pin_maxwell,
          "allencahn": W.pin_allencahn, "elasticity": W.pin_elasticity, "swe": W.pin_swe, "nsf2d": W.pin_nsf2d}


def _rows(case):
    return {r["n"]: r for r in PINS[case]["oracle"]}


def _sig5(a, b):
    """a (computed) equals b (printed with 5 significant digits) up to the last printed digit."""
    return abs(a - b) <= 1.01e-4 * abs(b)


@pytest.mark.parametrize("case", sorted(PINS))
def test_p8_stored_n512_equals_printed_values(case):
    rows = _rows(case)
    if 512 not in rows:
        pytest.skip(f"{case}: N = 512 row not generated yet (make_paper_pins.py)")
    paper = PINS[case]["paper_N512"]
    for field, (linf, l2) in rows[512]["fields"].items():
        p_linf, p_l2 = paper[field]
        assert _sig5(l2, p_l2), f"{case}.{field}: rel L2 {l2:.5e} vs printed {p_l2:.4e} ({paper['cite']})"
        assert _sig5(linf, p_linf), f"{case}.{field}: rel Linf {linf:.5e} vs printed {p_linf:.4e} ({paper['cite']})"


def _errors(case, n):
    w = MAKERS[case](n)
    g = oracle.OracleGrid.from_workload(w)
    if g.n_aux:
        g.set_aux(w.aux_fields())
    g.init_from_U(w.initial_U())
    g.step(w.steps)
    U = g.read_U()
    _, t = g.time()
    Ue = g.exact_U(t)
    g.close()
    out = []
    for k in range(U.shape[0]):
        e = U[k] - Ue[k]
        out.append((float(np.abs(e).max() / np.abs(Ue[k]).max()), float(np.sqrt((e * e).sum() / (Ue[k] * Ue[k]).sum()))))
    return out


@pytest.mark.parametrize("case", sorted(PINS))
def test_p8_live_n64_matches_stored_row(case):
    e = _errors(case, 64)
    stored = _rows(case)[64]["fields"]
    if case == "burgers":
        live = {"u": e[0]}
    elif case in ("euler", "nsf2d"):
        live = {"rho": e[0], "E": e[3], "rhou": (math.hypot(e[1][0], e[2][0]), math.hypot(e[1][1], e[2][1]))}
    elif case == "allencahn":
        live = {"phi": e[0]}
    elif case == "elasticity":
        rss = lambda ks, j: math.sqrt(sum(e[k][j] ** 2 for k in ks))
        live = {"F": (rss(range(4), 0), rss(range(4), 1)), "v": (rss((4, 5), 0), rss((4, 5), 1))}
    elif case == "urf":
        live = {"E": e[0], "S": (math.hypot(e[1][0], e[2][0]), math.hypot(e[1][1], e[2][1]))}
    elif case == "maxwell":
        live = {"Ez": e[0], "Hx": e[1], "Hy": e[2]}
    elif case == "swe":
        live = {"h": e[0], "hu": (math.hypot(e[1][0], e[2][0]), math.hypot(e[1][1], e[2][1]))}
    else:
        live = {"c": e[0]}
    for field, (linf, l2) in stored.items():
        assert live[field][0] == pytest.approx(linf, rel=1e-9)
        assert live[field][1] == pytest.approx(l2, rel=1e-9)


@pytest.mark.parametrize("case", sorted(PINS))
def test_p11_convergence_order_in_paper_band(case):
    rows = _rows(case)
    ns = sorted(rows)
    if len(ns) < 3:
        pytest.skip("need three resolutions")
    for field in rows[ns[0]]["fields"]:
        l2 = [rows[n]["fields"][field][1] for n in ns]
        slope = -np.polyfit(np.log2(ns), np.log2(l2), 1)[0]          # EOC = -LSQ slope
        assert 1.70 <= slope <= 2.51 + 0.35, f"{case}.{field}: L2 order {slope:.2f}"   # ADR's early rows are pre-asymptotic (2.8 pairwise, L510)


def test_nsf2d_orders_through_the_printed_n512_point():
    """Compressible NSF 2D, the paper's running example (reading A24: mu = K = 0.01 non-dimensional).
    The printed EOC is the least-squares slope over N = 64 ... 512 (L514).  Through the oracle's stored errors at N = 64, 128, 256
    and the PRINTED N = 512 error, that slope equals each of the six printed orders to their two decimals -- so the oracle's lower
    rows lie on the paper's convergence line (a wrong viscous or heat-flux term moves them by tens of percent, i.e. the slope by
    > 0.05).  The N = 512 row itself (131 072 steps) is checked digit by digit by test_p8_stored_n512_equals_printed_values."""
    rows = _rows("nsf2d")
    paper = PINS["nsf2d"]["paper_N512"]
    for field, eocs in paper["eoc"].items():
        for j in (0, 1):
            ys = [rows[n]["fields"][field][j] for n in (64, 128, 256)] + [paper[field][j]]
            slope = -np.polyfit(np.log2([64, 128, 256, 512]), np.log2(ys), 1)[0]
            assert abs(slope - eocs[j]) <= 0.0051, (field, j, slope, eocs[j])
