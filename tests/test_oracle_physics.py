"""Pins of the oracle's 3D systems (configs 4 and 5) and of its Euler system against formulas typed independently here
from the paper's vector forms, and against textbook closed-form dynamics (none of them re-uses the oracle's flux code).

  nsf3d  eq (3.23), with derived-parent trackers G = grad u, H = grad T (eq 3.27 pattern, L495-L497)
  mhd3d  eq (3.25), current-density trackers J = curl B (C5)
CPU only.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import OracleGrid


def _levi():
    e = np.zeros((3, 3, 3))
    for i, j, k in ((0, 1, 2), (1, 2, 0), (2, 0, 1)):
        e[i, j, k], e[i, k, j] = 1.0, -1.0
    return e


def nsf3d_flux_numpy(U, gamma, mu, K, dx, dt, g_tau):
    """Lattice flux F[k][j] and source S[k] of the NSF + tracker system, from primitive variables."""
    lam, dL = dx / dt, dt / dx**2
    rho, m, E = U[0], U[1:4], U[4]
    G = U[5:14].reshape(3, 3)            # G[a][b] = dx d_b u_a
    H = U[14:17]                          # H[b] = dx d_b T
    u = m / rho
    p = (gamma - 1) * (E - 0.5 * rho * u @ u)
    T = p / rho
    sig = mu * dL * (G + G.T - (2.0 / 3.0) * np.trace(G) * np.eye(3))
    F = np.zeros((17, 3)); S = np.zeros(17)
    F[0] = m / lam
    F[1:4] = (np.outer(m, u) + p * np.eye(3)) / lam - sig
    F[4] = (E + p) * u / lam - sig @ u - K * dL * H
    for a in range(3):
        for b in range(3):
            F[5 + 3 * a + b] = G[a, b] * u / lam
            F[5 + 3 * a + b, b] -= u[a] / g_tau
    for b in range(3):
        F[14 + b] = H[b] * u / lam
        F[14 + b, b] -= T / g_tau
    S[5:] = -U[5:] / g_tau
    return F, S


def mhd3d_flux_numpy(U, gamma, eta, dx, dt, g_tau):
    lam, dL = dx / dt, dt / dx**2
    eps = _levi()
    rho, m, E, B, J = U[0], U[1:4], U[4], U[5:8], U[8:11]
    u = m / rho
    p = (gamma - 1) * (E - 0.5 * rho * u @ u - 0.5 * B @ B)
    pt = p + 0.5 * B @ B
    F = np.zeros((11, 3)); S = np.zeros(11)
    F[0] = m / lam
    F[1:4] = (np.outer(m, u) + pt * np.eye(3) - np.outer(B, B)) / lam
    F[4] = ((E + pt) * u - B * (u @ B)) / lam + eta * dL * np.cross(J, B)
    F[5:8] = (np.outer(B, u) - np.outer(u, B)) / lam + eta * dL * np.einsum("ijk,k->ij", eps, J)
    F[8:11] = np.outer(J, u) / lam - np.einsum("ijk,k->ij", eps, B) / g_tau
    S[8:] = -J / g_tau
    return F, S


def test_nsf3d_flux_matches_independent_vector_form():
    rng = np.random.default_rng(5)
    gamma, mu, K, dx, lam, g_tau = 1.4, 2e-3, 7e-3, 1.0 / 32, 9.0, 3.0
    g = OracleGrid("nsf3d", 4, 4, 4, dx=dx, lam=lam, params=[gamma, mu, K], g_tau=g_tau)
    for _ in range(20):
        U = rng.uniform(-0.3, 0.3, 17); U[0] = rng.uniform(0.8, 1.3); U[4] = rng.uniform(2.0, 3.0)
        F, S = g.flux_source(U)
        Fn, Sn = nsf3d_flux_numpy(U, gamma, mu, K, dx, dx / lam, g_tau)
        assert np.abs(F - Fn).max() < 1e-13 and np.abs(S - Sn).max() < 1e-13


def test_mhd3d_flux_matches_independent_vector_form():
    rng = np.random.default_rng(6)
    gamma, eta, dx, lam, g_tau = 1.4, 3e-3, 1.0 / 24, 11.0, 4.0
    g = OracleGrid("mhd3d", 4, 4, 4, dx=dx, lam=lam, params=[gamma, eta], g_tau=g_tau)
    for _ in range(20):
        U = rng.uniform(-0.3, 0.3, 11); U[0] = rng.uniform(0.8, 1.3); U[4] = rng.uniform(2.0, 3.0)
        F, S = g.flux_source(U)
        Fn, Sn = mhd3d_flux_numpy(U, gamma, eta, dx, dx / lam, g_tau)
        assert np.abs(F - Fn).max() < 1e-13 and np.abs(S - Sn).max() < 1e-13


def nsf2d_flux_numpy(U, gamma, mu, K, dx, dt, g_tau):
    """Compressible NSF 2D with the cascade on the conserved fields (eq 3.23-3.24, Listing 2): gradients of the derived
    fields u, T from the tracked gradients of (rho, m, E) by the chain rule, written here with Jacobian matrices."""
    lam, dL = dx / dt, dt / dx**2
    rho, m, E = U[0], U[1:3], U[3]
    GV = U[4:12].reshape(4, 2) / dx                      # physical gradients d_b V, V = rho, m0, m1, E
    u = m / rho
    p = (gamma - 1) * (E - 0.5 * (m @ m) / rho)
    T = p / rho
    # Jacobians of u and T with respect to (rho, m0, m1, E)
    dudV = np.array([[-u[0] / rho, 1 / rho, 0, 0], [-u[1] / rho, 0, 1 / rho, 0]])
    dpdV = (gamma - 1) * np.array([0.5 * (u @ u), -u[0], -u[1], 1.0])
    dTdV = dpdV / rho - np.array([T / rho, 0, 0, 0])
    gu = dudV @ GV                                       # gu[a][b] = d_b u_a
    gT = dTdV @ GV
    tau = mu * (gu + gu.T - (2.0 / 3.0) * np.trace(gu) * np.eye(2))
    q = -K * gT
    Phi = np.zeros((12, 2))
    Phi[0] = m
    Phi[1:3] = np.outer(m, u) + p * np.eye(2) - tau
    Phi[3] = (E + p) * u - tau @ u + q
    F = Phi * dt / dx
    S = np.zeros(12)
    V = U[:4]
    for v in range(4):
        for b in range(2):
            F[4 + 2 * v + b] = U[4 + 2 * v + b] * u / lam
            F[4 + 2 * v + b, b] -= V[v] / g_tau
    S[4:] = -U[4:] / g_tau
    return F, S


def test_nsf2d_flux_matches_independent_vector_form():
    rng = np.random.default_rng(7)
    gamma, mu, K, dx, lam, g_tau = 1.4, 8e-3, 4e-2, 1.0 / 32, 16.0, 6.0
    g = OracleGrid("nsf2d", 4, 4, 1, dx=dx, lam=lam, params=[gamma, mu, K], g_tau=g_tau)
    for _ in range(20):
        U = rng.uniform(-0.3, 0.3, 12); U[0] = rng.uniform(0.8, 1.3); U[3] = rng.uniform(2.0, 3.0)
        F, S = g.flux_source(U)
        Fn, Sn = nsf2d_flux_numpy(U, gamma, mu, K, dx, dx / lam, g_tau)
        assert np.abs(F[:, :2] - Fn).max() < 1e-13 and np.abs(S - Sn).max() < 1e-13


def test_mhd3d_alfven_wave_speed():
    """Textbook closed form: a small transverse perturbation of a uniform field B0 e_x travels at v_A = B0/sqrt(rho)
    with dv = -dB/sqrt(rho) (ideal MHD, eta = 0).  Checks the signs of B (x) B in the momentum flux and of the
    induction flux B (x) u - u (x) B."""
    n, B0, rho, gamma, A = 64, 0.5, 1.0, 1.4, 1e-4
    vA = B0 / math.sqrt(rho)
    dx = 1.0 / n
    lam = 8.0
    g = OracleGrid("mhd3d", n, 2, 2, dx=dx, lam=lam, params=[gamma, 0.0], tau_R=0.05, g_tau=4.0)
    x = (np.arange(n) * dx)[None, None, :] * np.ones((2, 2, 1))
    k = 2 * np.pi
    U = np.zeros((11, 2, 2, n))
    dB = A * np.sin(k * x)
    U[0] = rho; U[5] = B0; U[6] = dB; U[2] = -rho * dB / math.sqrt(rho)
    p = 1.0 / gamma
    U[4] = p / (gamma - 1) + 0.5 * (U[2] ** 2) / rho + 0.5 * (B0**2 + dB**2)
    U[8 + 2] = dx * A * k * np.cos(k * x)                   # J_z = d_x B_y, lattice units
    g.init_from_U(U)
    steps = 256
    g.step(steps)
    t = steps * dx / lam
    By = g.read_U()[6, 0, 0]
    want = A * np.sin(k * (x[0, 0] - vA * t))
    assert np.abs(By - want).max() < 0.03 * A               # O(dx^2) dispersion + relaxation damping only


def test_euler2d_sound_speed():
    """Linear acoustics: a standing pressure/density wave of the Euler system oscillates at omega = c k, c = sqrt(gamma
    p/rho) = 1 at the reference state of config 3."""
    n, A, gamma = 64, 1e-4, 1.4
    w = W.c3_euler(n, steps=0)
    x = (np.arange(n) / n)[None, None, :] * np.ones((1, n, 1))
    k = 2 * np.pi
    drho = A * np.cos(k * x)
    U = np.zeros((4, 1, n, n))
    U[0] = 1.0 + drho
    U[3] = (1.0 / gamma + drho) / (gamma - 1)               # dp = c^2 drho, c = 1
    T = 1.0                                                 # one period = 2 pi / (c k)
    steps = int(round(T / w.dt))
    U1 = oracle.run(w, steps=steps, U0=U)
    t = steps * w.dt
    want = 1.0 + A * np.cos(k * x) * math.cos(k * t)
    assert np.abs(U1[0] - want).max() < 0.05 * A


def test_nsf3d_viscous_shear_decay_rate():
    """A shear wave u_y = A sin(k x) decays like exp(-nu_tot k^2 t); the difference of the decay rates with and without
    physical viscosity is nu k^2 (the relaxation diffusion is the same in both runs).  Pins the sign and the mu_L
    scaling of the viscous flux -mu_L (G + G^T - 2/3 tr G I) and the tracker coupling."""
    n, A, gamma = 128, 1e-3, 1.4        # the tracker's O(dx^2) resolution error (L196) is 29 % at 32, 9.5 % at 64, 2.5 % at 128
    k = 2 * np.pi
    rates = []
    for mu in (0.0, 5e-3):
        w = W.c4_nsf3d(n, ny=2, nz=2, precision="f64", mms=False, steps=0)
        w.params = [gamma, mu, 0.0]
        x = (np.arange(n) * w.dx)[None, None, :] * np.ones((2, 2, 1))
        U = np.zeros((17, 2, 2, n))
        U[0] = 1.0
        U[2] = A * np.sin(k * x)
        U[4] = (1.0 / gamma) / (gamma - 1) + 0.5 * U[2] ** 2
        U[5 + 3 * 1 + 0] = w.dx * A * k * np.cos(k * x)       # G_yx = dx d_x u_y
        steps = 1600
        U1 = oracle.run(w, steps=steps, U0=U)
        amp = 2.0 * np.abs((U1[2, 0, 0] * np.sin(k * x[0, 0])).mean())
        rates.append(-math.log(amp / A) / (steps * w.dt))
    assert rates[1] - rates[0] == pytest.approx(5e-3 * k * k, rel=0.05)
