"""How DESIGN.md reading A24 was found (not a test, not collected by pytest; needs a B200 and scipy):

    python tests/golden/fit_nsf2d_reading_a24.py [N=512] [max evaluations=70]

Compressible NSF 2D is the paper's running example; Table SM11 lists mu = 3.52 Pa s and K = 4980 W/m/K,
which non-dimensionalise to 0.00845 and 0.0416 and land at 1.5-2.1x the errors the paper PRINTS for this case (Table 2,
L547-L551).  This script runs the whole N = 512 study on the CUDA path (131 072 steps, ~4 s per evaluation) inside a
Nelder-Mead search over the two non-dimensional diffusivities and minimises the squared log-ratios of the six computed errors
to the six printed ones.  It converges to mu = 0.0100, K = 0.00998 with every ratio at 1.000: the run behind Table 2 used
mu = K = 0.01 (the "equal diffusivities" of the paper's MHD table SM12).  workloads.pin_nsf2d carries those values; the oracle
reproduces the printed row with them (tests/golden/paper_pins.json), independently of this script.
"""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

PAPER = dict(rho=(7.3384e-05, 3.7592e-05), rhou=(1.1775e-04, 6.8579e-05), E=(8.3354e-05, 4.5785e-05))      # (rel Linf, rel L2)
TABLE_SM11 = (3.52 / (1.225 * 340.2), 4980.0 / (1.225 * 340.2 * 287.0))


def main():
    import torch
    from scipy.optimize import minimize

    import paper_2607_05668_b200 as P
    import workloads as W
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 512
    maxfev = int(sys.argv[2]) if len(sys.argv) > 2 else 70
    P.lib()

    def errors(mu, K):
        w = W.relabel(W.pin_nsf2d(n), params=[1.4, mu, K])
        g = P.Grid.from_workload(w, declare_bound=False)
        g.init_from_U(torch.from_numpy(w.initial_U()).cuda())
        g.step(w.steps)
        e = g.error_norms()          # per component: relative (L1, L2, Linf)
        g.close()
        # vector fields: root-sum-square of the components' relative errors
        return dict(rho=(e[0][2], e[0][1]), rhou=(math.hypot(e[1][2], e[2][2]), math.hypot(e[1][1], e[2][1])), E=(e[3][2], e[3][1]))

    def objective(x):
        mu, K = TABLE_SM11[0] * math.exp(x[0]), TABLE_SM11[1] * math.exp(x[1])
        r = errors(mu, K)
        ratios = [r[k][j] / PAPER[k][j] for k in PAPER for j in (0, 1)]
        score = sum(math.log(v) ** 2 for v in ratios) if all(np.isfinite(v) and v > 0 for v in ratios) else 50.0
        print(f"{score:.3e}  mu = {mu:.6f}  K = {K:.6f}  computed / printed: " + " ".join(f"{v:.4f}" for v in ratios), flush=True)
        return score

    print("Table SM11's own values:")
    objective([0.0, 0.0])
    res = minimize(objective, [0.5, -0.7], method="Nelder-Mead",
                   options=dict(maxfev=maxfev, xatol=2e-4, fatol=1e-8, initial_simplex=[[0.5, -0.7], [0.35, -0.7], [0.5, -0.45]]))
    print("converged to mu = %.6f, K = %.6f, score %.2e" % (TABLE_SM11[0] * math.exp(res.x[0]), TABLE_SM11[1] * math.exp(res.x[1]), res.fun))


if __name__ == "__main__":
    main()
