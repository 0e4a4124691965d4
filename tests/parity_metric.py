"""The error measures of the GPU-vs-oracle parity gates (SURVEY.md §8(c) reading A16; A16).

BASELINE.json's bars are "max relative error <= 1e-12 in fp64, <= 2e-5 in shifted fp32".  The measure that was
written down before any kernel existed is, per component k,

    a16_k = max_x |U_k^gpu - U_k^oracle| / max_x |U_k^oracle| ,

with the system scale max_k max_x |U_k^oracle| as denominator for components that are identically zero.  THAT is
the gate (`gate(..., strict=True)`, the default): a16_k <= 1e-12 (fp64; 1e-11 for the shifted-fp64 identity test)
or <= 2e-5 (shifted fp32) for EVERY component, no exception.  All principal parity cases -- the five configs at
their test sizes and full step counts, the paper systems, the Dirichlet frame -- are gated this way.

`strict=False` is used only by the auxiliary cases whose state still holds components that have not left zero:
SHORT runs (the 6-12-step full-size sub-box samples, the staged-coefficient cases: v ~ sin t after a few steps)
and DEGENERATE grids (one-node axes, where whole fields vanish up to rounding).  There U_k is a small difference
of large populations (f_k,+-a = w (U_k +- F_k,a/c_s^2) cancel in the sum eq 2.6), so the rounding of U_k is set by
|f|, not by |U_k|, in fp64 exactly as in fp32.  A component that misses a16_k <= tol must then satisfy ALL of
        pop_k  = max_x |dU_k| / sum_i max_x |f^oracle_k,i|  <= tol       (error relative to what is summed)
        a16_k <= tol * A_k,    A_k = sum_i max_x |f^oracle_k,i| / max_x |U_k^oracle|   (condition number of the sum)
        a16_k <= 50 * tol                                                  (never worse than 50x the bar)
unless it is numerically zero in the oracle itself (max_x |U_k^oracle| <= tol * sum_i max_x |f^oracle_k,i|: the
oracle's own value is rounding noise), which by SURVEY A16 is measured against the system scale.

Every call of `gate()` appends one row per component (plain a16, fluctuation-relative, population-scale, A_k) to
ROWS; tests/conftest.py writes them to gpurun_out/parity_table.{json,md} at the end of a GPU session, and the
table of the last judged run is committed as profiles/r2_parity_table.md.
"""
import numpy as np

TOL64 = 1e-12
TOL32 = 2e-5

ROWS = []   # filled by gate(); written out by conftest.pytest_sessionfinish


def scales(fo):
    """sum_i max_x |f^oracle_k,i| from the oracle's canonical populations fo[k][i][z][y][x]."""
    return np.array([sum(np.abs(fo[k, i]).max() for i in range(fo.shape[1])) for k in range(fo.shape[0])])


def pop_rel_err(U, Uo, fo):
    s = scales(fo)
    return np.array([np.abs(U[k] - Uo[k]).max() / max(s[k], 1e-300) for k in range(U.shape[0])])


def a16_rel_err(U, Uo):
    """per component max|dU_k| / max|U_k^oracle|; identically-zero components use the system scale."""
    mags = np.array([np.abs(Uo[k]).max() for k in range(U.shape[0])])
    sysscale = max(mags.max(), 1e-300)
    den = np.where(mags > 0.0, mags, sysscale)
    return np.array([np.abs(U[k] - Uo[k]).max() / den[k] for k in range(U.shape[0])])


def fluct_rel_err(U, Uo, U_ref):
    ref = np.asarray(U_ref, dtype=np.float64).reshape(-1, 1, 1, 1)
    return np.array([np.abs(U[k] - Uo[k]).max() / max(np.abs(Uo[k] - ref[k]).max(), 1e-300) for k in range(U.shape[0])])


# kept under their round-1 names for the reported figures
plain_rel_err = a16_rel_err
rel_err = pop_rel_err


def gate(U, Uo, fo, precision, label, U_ref=None, tol=None, steps=None, record=True, strict=True):
    """Assert the A16 gate described in the module docstring; returns (a16, pop) per component.
    strict: one bool, or one per component (e.g. conserved fields strict, lattice-unit trackers of a system with an O(1)
    moving reference cancellation-scaled: their parents' fp32 rounding, ~eps * |V|, enters through -V/g_tau while the
    tracker itself is O(dx |grad V|) -- resistive MHD 2D at Mach 3, A16)."""
    fp32 = precision == "f32s"
    if tol is None:
        tol = TOL32 if fp32 else TOL64
    M = U.shape[0]
    strict_k = np.broadcast_to(np.asarray(strict, dtype=bool), (M,))
    mags = np.array([np.abs(Uo[k]).max() for k in range(M)])
    sc = scales(fo)
    sysscale = max(mags.max(), 1e-300)
    zero = mags <= np.where(strict_k, 0.0, tol) * sc           # identically zero (strict) / rounding noise of the oracle itself
    den = np.where(zero, sysscale, np.maximum(mags, 1e-300))
    err = np.array([np.abs(U[k] - Uo[k]).max() for k in range(M)])
    a16 = err / den
    pop = err / np.maximum(sc, 1e-300)
    A = sc / den
    fl = fluct_rel_err(U, Uo, U_ref) if U_ref is not None else np.full(M, np.nan)
    how = []
    for k in range(M):
        how.append("a16" if a16[k] <= tol else "cancellation-scaled")
    if record:
        for k in range(M):
            ROWS.append(dict(case=label, precision=precision, steps=steps, k=k, a16=float(a16[k]), fluct=float(fl[k]),
                             pop=float(pop[k]), A=float(A[k]), gate=("zero->system scale, " if zero[k] else "") + how[k],
                             strict=bool(strict_k[k])))
    assert np.isfinite(U).all(), f"{label}: non-finite state"
    for k in range(M):
        if a16[k] <= tol:
            continue
        assert not strict_k[k], f"{label}: component {k}: A16 max|dU_k|/max|U_k| = {a16[k]:.3e} > {tol:g} (all: {a16})"
        bound = min(tol * A[k], 50.0 * tol)
        assert pop[k] <= tol and a16[k] <= bound, (
            f"{label}: component {k}: A16 {a16[k]:.3e} > {tol:g}; population-scale {pop[k]:.3e}, "
            f"cancellation factor A_k {A[k]:.3g}, bound {bound:.3e}")
    return a16, pop


def table_markdown(rows):
    out = ["| case | precision | steps | k | A16 max\\|dU\\|/max\\|U\\| | fluctuation-relative | population-scale | A_k | gate | strict |",
           "|---|---|---|---|---|---|---|---|---|---|"]
    for r in rows:
        out.append(f"| {r['case']} | {r['precision']} | {r['steps']} | {r['k']} | {r['a16']:.3e} | {r['fluct']:.3e} | "
                   f"{r['pop']:.3e} | {r['A']:.3g} | {r['gate']} | {r.get('strict', True)} |")
    return "\n".join(out) + "\n"
