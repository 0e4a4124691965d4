"""Pins of the three systems round 2 added to the oracle (CPU only):
  swe2d_bathy  shallow water over a bed, eq (3.5)-(3.6), PAPER.md:L351-L359 (bed slope = prescribed per-node field)
  hcnsf3d      homogenized NSF, eq (3.27); listing SM4.12 L1017-L1143 (alpha, u_s prescribed)
  mhd2d        resistive MHD 2D with Powell source, eq (3.25); legible parts of listing SM4.11

P1 (equilibrium moments), P3 (Lax-Friedrichs collapse at omega = 1), P10 (manufactured forcing against a finite-difference
residual of Q_exact and Phi(Q_exact) -- independent of the jets) and P13: a brute-force NumPy step whose fluxes are typed
from the paper's EXPANDED LISTINGS (chi sub-expressions of SM4.12; the printed Phi_{1,0}, Phi_{1,1}, induction, tracker and
source components of SM4.11), i.e. a different algebraic form than the vector form the oracle is written in.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from brute_force import init_equilibrium, moments, step as bf_step

rng0 = np.random.default_rng(20261105)


# ------------------------------------------------------------------------------------------------ listings
def hcnsf_listing(U, A, gamma, mu, kappa, eta, tau_grad):
    """SM4.12 in the paper's own sub-expressions chi_i, PHYSICAL trackers.  U in THIS build's order
    (rho, m0, m1, m2, E, Gu00, Gu11, Gu22, Su01, Su02, Su12, Gaux0, Gaux1, Gaux2); A = (alpha, us0, us1, us2).
    Returns (Phi[k][a], S[k]).  The energy flux listing is cut in the source (L1100): eq (3.27) is typed instead."""
    rho, m0, m1, m2, E, G00, G11, G22, S01, S02, S12, X0, X1, X2 = U
    al, us0, us1, us2 = A
    c0 = m0 ** 2; c1 = 1 / rho; c2 = 3 * c1 / 2; c3 = al * mu; c4 = 4 * c3 / 3; c5 = -E; c6 = E * gamma; c7 = m2 ** 2
    c8 = c1 / 2; c9 = c7 * c8; c10 = c0 * c8; c11 = -c10 * gamma; c12 = m1 ** 2; c13 = c12 * c8; c14 = -c13 * gamma
    c15 = -c9 * gamma; c16 = 2 * c3 / 3
    c17 = G22 * c16 + c11 + c14 + c15 + c5 + c6 + c9
    c18 = G11 * c16 + c13
    c19 = 2 * c3
    c20 = -S01 * c19 + c1 * m0 * m1
    c21 = -S02 * c19 + c1 * m0 * m2
    c22 = G00 * c16 + c10
    c23 = -S12 * c19 + c1 * m1 * m2
    c24 = al * kappa; c25 = 1 / rho ** 2; c27 = c25 / 2
    c28 = c1 * m0; c29 = G00 * c28; c30 = c1 * m1; c31 = S01 * c30; c32 = c1 * m2; c33 = S02 * c32
    c36 = G11 * c30; c37 = S01 * c28; c38 = S12 * c32; c41 = G22 * c32; c42 = S02 * c28; c43 = S12 * c30
    c45 = 1 / tau_grad; c46 = c1 * c45; c47 = c27 * c45; c48 = c0 * c47; c49 = c12 * c47; c50 = c47 * c7
    c51 = E * c46 - c46 * c6 + c48 * gamma - c48 + c49 * gamma - c49 + c50 * gamma - c50
    c52 = c45 * c8; c53 = -c52 * m1; c54 = -c52 * m0; c55 = -c52 * m2
    P = {}
    P[0] = [m0, m1, m2]
    P[1] = [-G00 * c4 + c0 * c2 + c17 + c18, c20, c21]
    P[2] = [c20, -G11 * c4 + c12 * c2 + c17 + c22, c23]
    P[3] = [c21, c23, -G22 * c4 + c11 + c14 + c15 + c18 + c2 * c7 + c22 + c5 + c6]
    # energy: (E + p) u - alpha tau.u - alpha kappa G^aux, eq (3.27)
    u = [c28, c30, c32]
    p = (gamma - 1) * (E - (c0 + c12 + c7) * c8)
    tr = G00 + G11 + G22
    sym = [[G00, S01, S02], [S01, G11, S12], [S02, S12, G22]]
    tau = [[mu * (2 * sym[a][b] - (2 / 3 * tr if a == b else 0)) for b in range(3)] for a in range(3)]
    X = [X0, X1, X2]
    P[4] = [(E + p) * u[j] - al * sum(tau[j][b] * u[b] for b in range(3)) - c24 * X[j] for j in range(3)]
    P[5] = [-c28 * c45 + c29, G00 * c30, G00 * c32]                     # paper's Q10 = G_u00
    P[6] = [G11 * c28, -c30 * c45 + c36, G11 * c32]                     # paper's Q5
    P[7] = [G22 * c28, G22 * c30, -c32 * c45 + c41]                     # paper's Q6
    P[8] = [c37 + c53, c31 + c54, S01 * c32]                            # paper's Q11
    P[9] = [c42 + c55, S02 * c30, c33 + c54]                            # paper's Q12
    P[10] = [S12 * c28, c43 + c55, c38 + c53]                           # paper's Q13
    P[11] = [X0 * c28 + c51, X0 * c30, X0 * c32]                        # paper's Q7..Q9
    P[12] = [X1 * c28, X1 * c30 + c51, X1 * c32]
    P[13] = [X2 * c28, X2 * c30, X2 * c32 + c51]
    S = [0 * rho,
         -al * us0 * rho / eta + al * m0 / eta + us0 * rho / eta - m0 / eta,
         -al * us1 * rho / eta + al * m1 / eta + us1 * rho / eta - m1 / eta,
         -al * us2 * rho / eta + al * m2 / eta + us2 * rho / eta - m2 / eta,
         (-al * us0 * m0 - al * us1 * m1 - al * us2 * m2 + al * (c0 + c12 + c7) / rho + us0 * m0 + us1 * m1 + us2 * m2
          - (c0 + c12 + c7) / rho) / eta]
    S += [-U[k] / tau_grad for k in range(5, 14)]
    return [P[k] for k in range(14)], S


def mhd2d_listing(U, gamma, mu, K, eta, tau_grad):
    """SM4.11, PHYSICAL trackers, THIS build's order (rho, m0, m1, E, B0, B1, G_{V,b} for V = rho, m0,
    m1, E, B0, B1).  Typed from the print: Phi_{1,0}, Phi_{1,1} (and their x<->y images), induction, trackers, sources.
    The energy flux print is garbled: eq (3.25) L476 is typed instead."""
    rho, m0, m1, E, B0, B1 = U[:6]
    Gr, Gm0, Gm1, GE, GB0, GB1 = [(U[6 + 2 * v], U[7 + 2 * v]) for v in range(6)]
    z = 0 * rho
    P10 = (-B0 ** 2 * gamma / 2 - B1 ** 2 * gamma / 2 + B1 ** 2 + E * gamma - E + 4 * Gr[0] * mu * m0 / (3 * rho ** 2)
           - 2 * Gr[1] * mu * m1 / (3 * rho ** 2) - 4 * Gm0[0] * mu / (3 * rho) + 2 * Gm1[1] * mu / (3 * rho)
           - gamma * m0 ** 2 / (2 * rho) - gamma * m1 ** 2 / (2 * rho) + 3 * m0 ** 2 / (2 * rho) + m1 ** 2 / (2 * rho))
    P11 = (-B0 * B1 + Gr[0] * mu * m1 / rho ** 2 + Gr[1] * mu * m0 / rho ** 2 - Gm0[1] * mu / rho - Gm1[0] * mu / rho + m0 * m1 / rho)
    P21 = (-B0 ** 2 * gamma / 2 - B1 ** 2 * gamma / 2 + B0 ** 2 + E * gamma - E - 2 * Gr[0] * mu * m0 / (3 * rho ** 2)
           + 4 * Gr[1] * mu * m1 / (3 * rho ** 2) + 2 * Gm0[0] * mu / (3 * rho) - 4 * Gm1[1] * mu / (3 * rho)
           - gamma * m0 ** 2 / (2 * rho) - gamma * m1 ** 2 / (2 * rho) + m0 ** 2 / (2 * rho) + 3 * m1 ** 2 / (2 * rho))
    # energy flux from eq (3.25): (E + p_tot) u - B (u.B) - tau.u + q + eta (j x B), q = -K grad T, T = p/rho
    u = [m0 / rho, m1 / rho]
    B = [B0, B1]
    B2 = B0 ** 2 + B1 ** 2
    p = (gamma - 1) * (E - (m0 ** 2 + m1 ** 2) / (2 * rho) - B2 / 2)
    pt = p + B2 / 2
    du = [[(Gm0[b] - u[0] * Gr[b]) / rho for b in range(2)], [(Gm1[b] - u[1] * Gr[b]) / rho for b in range(2)]]
    dp = [(gamma - 1) * (GE[b] - u[0] * Gm0[b] - u[1] * Gm1[b] + (u[0] ** 2 + u[1] ** 2) / 2 * Gr[b] - B0 * GB0[b] - B1 * GB1[b]) for b in range(2)]
    dT = [(dp[b] - p / rho * Gr[b]) / rho for b in range(2)]
    div = du[0][0] + du[1][1]
    tau = [[mu * (du[a][b] + du[b][a] - (2 / 3 * div if a == b else 0)) for b in range(2)] for a in range(2)]
    jz = GB1[0] - GB0[1]
    jxB = [-jz * B1, jz * B0]
    uB = u[0] * B0 + u[1] * B1
    P3 = [(E + pt) * u[j] - B[j] * uB - (tau[j][0] * u[0] + tau[j][1] * u[1]) - K * dT[j] + eta * jxB[j] for j in range(2)]
    Phi = [[m0, m1, z], [P10, P11, z], [P11, P21, z], [P3[0], P3[1], z],
           [-GB0[0] * eta, B0 * m1 / rho - B1 * m0 / rho - GB0[1] * eta, z],                   # Phi_{4,0}, Phi_{4,1}
           [-B0 * m1 / rho + B1 * m0 / rho - GB1[0] * eta, -GB1[1] * eta, z]]                  # Phi_{5,0}, Phi_{5,1}
    V = [rho, m0, m1, E, B0, B1]
    for v, G in enumerate((Gr, Gm0, Gm1, GE, GB0, GB1)):                                       # Phi_{6..17}: G m/rho - delta V/tau_grad
        Phi.append([G[0] * m0 / rho - V[v] / tau_grad, G[0] * m1 / rho, z])
        Phi.append([G[1] * m0 / rho, G[1] * m1 / rho - V[v] / tau_grad, z])
    S = [z, -B0 * GB0[0] - B0 * GB1[1], -B1 * GB0[0] - B1 * GB1[1],
         -B0 * GB0[0] * m0 / rho - B0 * GB1[1] * m0 / rho - B1 * GB0[0] * m1 / rho - B1 * GB1[1] * m1 / rho,
         -GB0[0] * m0 / rho - GB1[1] * m0 / rho, -GB0[0] * m1 / rho - GB1[1] * m1 / rho]
    S += [-U[k] / tau_grad for k in range(6, 18)]
    return Phi, S


# ------------------------------------------------------------------------------------------------ helpers
def _bf(w, steps, lat, aux=None):
    """Brute-force run: lat(U list[, A]) -> (F lattice, S lattice)."""
    U = list(w.initial_U())
    mc = W.N_CONSERVED[w.system]
    omega = [1.0 / (0.5 + w.tau_R * w.dt)] * mc + [1.0 / (w.g_tau + 1.0)] * (w.m_total - mc)
    F, S = lat(U)
    f = init_equilibrium(U, F, w.dim)
    for _ in range(steps):
        Uc = moments(f)
        F, S = lat(Uc)
        f = bf_step(f, w.dim, omega, F, S)
    return np.stack(moments(f))


def _oracle(w, steps, A=None):
    g = oracle.OracleGrid.from_workload(w)
    if g.n_aux:
        g.set_aux(A if A is not None else w.aux_fields())
    g.init_from_U(w.initial_U())
    g.step(steps)
    U = g.read_U()
    g.close()
    return U


# ------------------------------------------------------------------------------------------------ P13
def test_p13_brute_force_swe_over_a_bed():
    """SM4.3 flux listing (L831) + the bed source of eq (3.6): S = (0, -g h d_0 z_b, -g h d_1 z_b)."""
    from brute_force import flux_swe_listing
    w = W.relabel(W.pin_swe(8), ny=6, mms_id=0)
    A = w.aux_fields()
    g, il, dt = w.params[0], 1.0 / w.lam, w.dt

    def lat(U):
        Phi = flux_swe_listing(U, g)
        return [[il * Phi[k][a] for a in range(3)] for k in range(3)], [0 * U[0], -dt * g * U[0] * A[0], -dt * g * U[0] * A[1]]

    assert np.abs(_oracle(w, 12) - _bf(w, 12, lat)).max() < 1e-15


def test_p13_brute_force_hcnsf_listing():
    """The chi-listing of SM4.12 against the oracle's vector form: stress coefficients 4/3, 2/3 and 2 alpha mu on the
    symmetric trackers, the halves of sym(I (x) u)/tau_grad, the temperature injection chi_51 = -T/tau_grad, the drag."""
    w = W.hcnsf3d(6, ny=5, nz=4, precision="f64")
    gamma, mu, kappa, eta = w.params
    A = w.aux_fields(0.3)
    il, dt, dx = 1.0 / w.lam, w.dt, w.dx
    tau_grad = w.g_tau * dt

    def lat(U):
        Up = list(U[:5]) + [U[k] / dx for k in range(5, 14)]             # lattice trackers -> physical gradients
        Phi, Sp = hcnsf_listing(Up, A, gamma, mu, kappa, eta, tau_grad)
        F = [[il * Phi[k][a] for a in range(3)] for k in range(5)] + [[il * dx * Phi[k][a] for a in range(3)] for k in range(5, 14)]
        S = [dt * Sp[k] for k in range(5)] + [dt * dx * Sp[k] for k in range(5, 14)]
        return F, S

    U = _oracle(w, 10, A)
    Ub = _bf(w, 10, lat)
    assert np.abs(U - Ub).max() < 1e-13 * np.abs(U).max()


def test_p13_brute_force_mhd2d_listing():
    w = W.relabel(W.pin_mhd2d(8), ny=6, mms_id=0)
    gamma, mu, K, eta = w.params
    il, dt, dx = 1.0 / w.lam, w.dt, w.dx
    tau_grad = w.g_tau * dt
    U0 = w.initial_U()
    x = (np.arange(w.nx) * dx)[None, None, :]
    y = (np.arange(w.ny) * dx)[None, :, None]
    U0[4] += 0.2 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y / (w.ny * dx))     # non-trivial B and grad B (div B != 0: Powell source active)
    U0[5] += 0.1 * np.cos(2 * np.pi * x)
    U0[14] = dx * 0.2 * 2 * np.pi * np.cos(2 * np.pi * x) * np.cos(2 * np.pi * y / (w.ny * dx))
    U0[16] = -dx * 0.1 * 2 * np.pi * np.sin(2 * np.pi * x) + 0 * y
    w = W.relabel(w, init=lambda _w: U0)

    def lat(U):
        Up = list(U[:6]) + [U[k] / dx for k in range(6, 18)]
        Phi, Sp = mhd2d_listing(Up, gamma, mu, K, eta, tau_grad)
        F = [[il * Phi[k][a] for a in range(3)] for k in range(6)] + [[il * dx * Phi[k][a] for a in range(3)] for k in range(6, 18)]
        S = [dt * Sp[k] for k in range(6)] + [dt * dx * Sp[k] for k in range(6, 18)]
        return F, S

    U = _oracle(w, 10)
    Ub = _bf(w, 10, lat)
    assert np.abs(U - Ub).max() < 1e-13 * np.abs(U).max()


# ------------------------------------------------------------------------------------------------ P1, P3
def _state(system):
    r = np.random.default_rng(11)
    if system == "swe2d_bathy":
        return np.array([0.9, 0.2, -0.1]), [9.81], np.array([0.3, -0.2])
    if system == "hcnsf3d":
        return np.concatenate([[1.2, 0.3, -0.2, 0.1, 3.0], 0.05 * r.standard_normal(9)]), [1.4, 1e-2, 2e-2, 0.1], np.array([0.6, 0.1, -0.2, 0.05])
    return np.concatenate([[1.2, 0.3, -0.2, 3.5, 0.4, -0.3], 0.05 * r.standard_normal(12)]), [1.4, 1e-2, 2e-2, 5e-3], np.zeros(1)


@pytest.mark.parametrize("system", ["swe2d_bathy", "hcnsf3d", "mhd2d"])
def test_p1_equilibrium_moments(system):
    """eq (2.8): sum_i f_eq = U_k, sum_i c_i f_eq = F_k for the flux the oracle forms (prescribed fields in)."""
    U, params, A = _state(system)
    dim = 3 if system == "hcnsf3d" else 2
    o = oracle.OracleGrid(system, 4, 4, 4 if dim == 3 else 1, 0.05, 6.0, params=params, g_tau=3.0)
    F, S = o.flux_source(U, A)
    feq = o.equilibrium(U, F)
    c, w_, cs2 = oracle.lattice(dim)
    assert np.allclose(feq.sum(1), U, rtol=1e-14, atol=1e-16)
    assert np.allclose(feq @ c.astype(float), F, rtol=1e-13, atol=1e-16)
    o.close()


@pytest.mark.parametrize("mk,kw", [(W.pin_swe, dict(n=8)), (W.hcnsf3d, dict(n=6, ny=5, nz=4, precision="f64")), (W.pin_mhd2d, dict(n=8))])
def test_p3_lax_friedrichs(mk, kw):
    """omega = 1 (L142): U_new = w0 U + w sum_a [U(x-e_a) + U(x+e_a)] - 1/2 sum_a [F_a(x+e_a) - F_a(x-e_a)] + s(x)...: one step of
    the oracle equals this finite-difference formula built from the oracle's pointwise flux (source added at the node)."""
    w = W.relabel(mk(**kw), mms_id=0)
    U0 = w.initial_U()
    A = w.aux_fields() if w.n_aux else None
    o = oracle.OracleGrid.from_workload(w, omega=1.0)
    if A is not None:
        o.set_aux(A)
    o.init_from_U(U0)
    o.step(1)
    U1 = o.read_U()
    m, D = w.m_total, w.dim
    F = np.zeros((m, 3) + U0.shape[1:]); S = np.zeros_like(U0)
    for idx in np.ndindex(U0.shape[1:]):
        Fi, Si = o.flux_source(U0[(slice(None),) + idx], None if A is None else A[(slice(None),) + idx])
        F[(slice(None), slice(None)) + idx] = Fi
        S[(slice(None),) + idx] = Si
    o.close()
    w0, w1 = (1 / 3, 1 / 6) if D == 2 else (1 / 4, 1 / 8)
    # post-collision populations carry w_i S of THEIR node: after streaming, node x holds w0 S(x) + w1 sum_a [S(x-e_a) + S(x+e_a)]
    want = w0 * (U0 + S)
    for a in range(D):
        ax = 3 - a                                   # array axis of coordinate a in U[k][z][y][x]
        want += w1 * (np.roll(U0 + S, 1, ax) + np.roll(U0 + S, -1, ax))
        want -= 0.5 * (np.roll(F[:, a], -1, ax) - np.roll(F[:, a], 1, ax))
    assert np.abs(U1 - want).max() < 1e-13 * np.abs(U1).max()


# ------------------------------------------------------------------------------------------------ P10
@pytest.mark.parametrize("mk", [W.pin_swe, W.pin_mhd2d])
def test_p10_mms_forcing_matches_fd_residual(mk):
    """eq (4.1): s = dt d_t Q + dx div F(Q_exact) - S(Q_exact) against central differences of the oracle's exact
    state and of its flux evaluated there (h = 1e-5); the bed slope handed to the flux is the workload's closed form."""
    w = mk(32)
    o = oracle.OracleGrid.from_workload(w)
    r = np.random.default_rng(5)
    k = 2 * np.pi
    for _ in range(6):
        t, x, y = r.uniform(0.1, 0.9), r.uniform(0, 1), r.uniform(0, 1)
        A = None
        if w.n_aux:
            Azb = w.mms_params[4]
            A = lambda xx, yy: np.array([Azb * k * np.cos(k * xx) * np.cos(k * yy), -Azb * k * np.sin(k * xx) * np.sin(k * yy)])
        h = 1e-5
        Q = lambda tt, xx, yy: o.exact_point(tt, xx, yy)
        Fl = lambda tt, xx, yy: o.flux_source(Q(tt, xx, yy), None if A is None else A(xx, yy))
        dQdt = (Q(t + h, x, y) - Q(t - h, x, y)) / (2 * h)
        dFx = (Fl(t, x + h, y)[0][:, 0] - Fl(t, x - h, y)[0][:, 0]) / (2 * h)
        dFy = (Fl(t, x, y + h)[0][:, 1] - Fl(t, x, y - h)[0][:, 1]) / (2 * h)
        want = w.dt * dQdt + w.dx * (dFx + dFy) - Fl(t, x, y)[1]
        got = o.mms_source(t, x, y)
        scale = np.abs(want).max()
        assert np.abs(got - want).max() < 2e-6 * scale, (w.system, got, want)
    o.close()


@pytest.mark.parametrize("mk", [W.pin_swe, W.pin_mhd2d])
def test_exact_fields_match_workload_inputs(mk):
    w = mk(16)
    o = oracle.OracleGrid.from_workload(w)
    assert np.abs(o.exact_U(0.0) - w.initial_U()).max() < 1e-13
    o.close()
