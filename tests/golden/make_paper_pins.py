"""Writes tests/golden/paper_pins.json: the oracle's errors on the Table 2 rows of the paper
that SURVEY.md Appendix A gives full recipes for, next to the values the paper prints.

Calls ONLY `oracle/` and `workloads/` (never the CUDA path).  Run from the repo root:
    python tests/golden/make_paper_pins.py            # N = 64,128,256,512; hours on 8 cores (the diffusive cases at N = 512)
The N = 512 rows are the pins (Table 2); the lower-N rows are fast
regression values for the default CPU test run (tests/test_oracle_paper_pins.py).
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import workloads as W  # noqa: E402

# values printed in PAPER.md Table 2 (double precision, N = 512, t = 1): (rel Linf, rel L2)
PAPER = {
    "burgers": {"u": (6.1175e-04, 8.5671e-05), "cite": "PAPER.md:L518"},
    "euler": {"E": (3.3385e-06, 1.8316e-06), "rho": (1.4401e-06, 6.8435e-07), "rhou": (3.2141e-06, 1.8745e-06),
              "cite": "PAPER.md:L519-L522 (row labels E, rho, rho u: SURVEY.md §8(c) A8)"},
    "adr": {"c": (2.2901e-04, 1.2680e-04), "cite": "PAPER.md:L540"},
    "allencahn": {"phi": (7.3196e-04, 7.8653e-04), "cite": "PAPER.md:L542"},
    "elasticity": {"F": (3.1874e-05, 2.8940e-05), "v": (6.4804e-05, 4.5664e-05), "cite": "PAPER.md:L536-L539"},
    "urf": {"E": (4.3449e-06, 2.1354e-06), "S": (9.6256e-06, 6.3943e-06), "cite": "PAPER.md:L527-L529"},
    "swe": {"h": (5.5560e-06, 2.3433e-06), "hu": (2.6837e-05, 2.0838e-05), "cite": "PAPER.md:L523-L526"},
    "nsf2d": {"rho": (7.3384e-05, 3.7592e-05), "rhou": (1.1775e-04, 6.8579e-05), "E": (8.3354e-05, 4.5785e-05),
              "eoc": {"rho": (1.91, 1.95), "rhou": (1.95, 1.99), "E": (1.98, 2.01)},
              "cite": "PAPER.md:L547-L551 (N = 512: 131 072 steps of 12 fields, ~1.6 h on 8 cores)"},
    "maxwell": {"Ez": (2.9956e-05, 2.9956e-05), "Hx": (1.0951e-04, 1.0951e-04), "Hy": (1.1587e-05, 1.1587e-05),
                "cite": "PAPER.md:L530-L535"},
}


def rel_errors(U, Ue):
    """per component (rel Linf, rel L2), PAPER.md:L504"""
    out = []
    for k in range(U.shape[0]):
        e = U[k] - Ue[k]
        out.append((float(np.abs(e).max() / np.abs(Ue[k]).max()), float(np.sqrt((e * e).sum() / (Ue[k] * Ue[k]).sum()))))
    return out


def run_case(case, n):
    w = {"burgers": W.pin_burgers, "euler": W.pin_euler, "adr": W.pin_adr, "urf": W.pin_urf, "maxwell": W.pin_maxwell,
         "allencahn": W.pin_allencahn, "elasticity": W.pin_elasticity, "swe": W.pin_swe, "nsf2d": W.pin_nsf2d}[case](n)
    g = oracle.OracleGrid.from_workload(w)
    if g.n_aux:
        g.set_aux(w.aux_fields())          # static bed slope
    g.init_from_U(w.initial_U())
    t0 = time.time()
    g.step(w.steps)
    wall = time.time() - t0
    U = g.read_U()
    _, t = g.time()
    e = rel_errors(U, g.exact_U(t))
    g.close()
    if case == "burgers":
        fields = {"u": e[0]}
    elif case == "nsf2d":
        fields = {"rho": e[0], "E": e[3],
                  "rhou": (float(np.hypot(e[1][0], e[2][0])), float(np.hypot(e[1][1], e[2][1])))}
    elif case == "euler":
        # vector field norm = root-sum-square of the components' relative norms
        fields = {"rho": e[0], "E": e[3],
                  "rhou": (float(np.hypot(e[1][0], e[2][0])), float(np.hypot(e[1][1], e[2][1])))}
    elif case == "allencahn":
        fields = {"phi": e[0]}
    elif case == "elasticity":
        rss = lambda ks, j: float(np.sqrt(sum(e[k][j] ** 2 for k in ks)))
        fields = {"F": (rss(range(4), 0), rss(range(4), 1)), "v": (rss((4, 5), 0), rss((4, 5), 1))}
    elif case == "urf":
        fields = {"E": e[0], "S": (float(np.hypot(e[1][0], e[2][0])), float(np.hypot(e[1][1], e[2][1])))}
    elif case == "maxwell":
        fields = {"Ez": e[0], "Hx": e[1], "Hy": e[2]}
    elif case == "swe":
        fields = {"h": e[0], "hu": (float(np.hypot(e[1][0], e[2][0])), float(np.hypot(e[1][1], e[2][1])))}
    else:
        fields = {"c": e[0]}
    return {"n": n, "steps": w.steps, "t_final": t, "wall_s": round(wall, 1), "fields": fields}


if __name__ == "__main__":
    # usage: make_paper_pins.py [case ...] [--sizes 64,128]   (--sizes: only these N, merged into the case's existing rows)
    args = sys.argv[1:]
    sizes = None
    if "--sizes" in args:
        i = args.index("--sizes")
        sizes = tuple(int(v) for v in args[i + 1].split(","))
        args = args[:i] + args[i + 2:]
    cases = args or ["burgers", "euler", "adr", "urf", "maxwell", "allencahn", "elasticity", "swe", "nsf2d"]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_pins.json")
    for case in cases:
        rows = []
        for n in (sizes or (64, 128, 256, 512)):
            r = run_case(case, n)
            print(case, r, flush=True)
            rows.append(r)
        out = json.load(open(path)) if os.path.exists(path) else {}       # re-read: another run may have written meanwhile
        if sizes and case in out:
            keep = [r for r in out[case]["oracle"] if r["n"] not in sizes]
            rows = sorted(keep + rows, key=lambda r: r["n"])
        out[case] = {"paper_N512": PAPER[case], "oracle": rows}
        json.dump(out, open(path, "w"), indent=1, sort_keys=True)
