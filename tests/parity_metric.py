"""The error measure of the GPU-vs-oracle parity gates (reading A16).

BASELINE.json's bars are "max relative error <= 1e-12 in fp64, <= 2e-5 in shifted fp32" and do not say
relative to what.  Reading: per component k,

    err_k = max_x |U_k^gpu - U_k^oracle| / scale_k,      scale_k = sum_i max_x |f^oracle_k,i|,

i.e. relative to the magnitude of the populations whose sum U_k is (eq 2.6).  scale_k >= max_x |U_k|, with
equality when the populations of k do not change sign; it differs for components that are small next to
their own flux (momentum in a fluid at rest: f_m,+-a = w (m +- p/(lambda c_s^2)) cancel in the sum), where
rounding of U_k is set by |f|, not by |U_k|.  The plain figure max|dU_k| / max|U_k| and the figure relative
to the fluctuation max|U_k - Q0_k| are reported beside it, not gated.
"""
import numpy as np


def scales(fo):
    """scale_k from the oracle's canonical populations fo[k][i][z][y][x]."""
    return np.array([sum(np.abs(fo[k, i]).max() for i in range(fo.shape[1])) for k in range(fo.shape[0])])


def rel_err(U, Uo, fo):
    s = scales(fo)
    return np.array([np.abs(U[k] - Uo[k]).max() / max(s[k], 1e-300) for k in range(U.shape[0])])


def plain_rel_err(U, Uo):
    return np.array([np.abs(U[k] - Uo[k]).max() / max(np.abs(Uo[k]).max(), 1e-300) for k in range(U.shape[0])])


def fluct_rel_err(U, Uo, U_ref):
    ref = np.asarray(U_ref, dtype=np.float64).reshape(-1, 1, 1, 1)
    return np.array([np.abs(U[k] - Uo[k]).max() / max(np.abs(Uo[k] - ref[k]).max(), 1e-300) for k in range(U.shape[0])])
