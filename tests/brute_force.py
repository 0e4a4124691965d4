"""Brute-force NumPy collide-and-stream step, written directly from the moment definitions
(eq 2.6, 2.7, 2.11 of PAPER.md) with explicit sums and np.roll -- pin P13 of SURVEY.md §8(c).

Independent of `oracle/` (own lattice tables, own streaming, own fluxes).  The fluxes are typed
from the paper's *expanded component listings* (SM4.2, SM4.3, SM4.7), i.e. a different algebraic
form than the primitive-variable form the oracle uses.
"""
import numpy as np

# Table SM1
LATTICES = {
    2: dict(c=[(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0)],
            w=[1 / 3, 1 / 6, 1 / 6, 1 / 6, 1 / 6], cs2=1 / 3),
    3: dict(c=[(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)],
            w=[1 / 4, 1 / 8, 1 / 8, 1 / 8, 1 / 8, 1 / 8, 1 / 8], cs2=1 / 4),
}


def flux_euler_listing(U, gamma):
    """SM4.2, PAPER.md:L819 (expanded component form). U[k] arrays; returns Phi[k][a] physical."""
    rho, m0, m1, E = U
    P10 = E * gamma - E - gamma * m0**2 / (2 * rho) - gamma * m1**2 / (2 * rho) + 3 * m0**2 / (2 * rho) + m1**2 / (2 * rho)
    P11 = m0 * m1 / rho
    P21 = E * gamma - E - gamma * m0**2 / (2 * rho) - gamma * m1**2 / (2 * rho) + m0**2 / (2 * rho) + 3 * m1**2 / (2 * rho)
    P30 = E * gamma * m0 / rho - gamma * m0**3 / (2 * rho**2) - gamma * m0 * m1**2 / (2 * rho**2) + m0**3 / (2 * rho**2) + m0 * m1**2 / (2 * rho**2)
    P31 = E * gamma * m1 / rho - gamma * m0**2 * m1 / (2 * rho**2) - gamma * m1**3 / (2 * rho**2) + m0**2 * m1 / (2 * rho**2) + m1**3 / (2 * rho**2)
    z = np.zeros_like(rho)
    return [[m0, m1, z], [P10, P11, z], [P11, P21, z], [P30, P31, z]]


def flux_swe_listing(U, g):
    """SM4.3."""
    h, q0, q1 = U
    z = np.zeros_like(h)
    return [[q0, q1, z], [g * h**2 / 2 + q0**2 / h, q0 * q1 / h, z], [q0 * q1 / h, g * h**2 / 2 + q1**2 / h, z]]


def flux_adr_listing(U, u0, u1, D, tau_grad):
    """SM4.7, PHYSICAL tracker G = grad c. Returns (Phi, S) physical."""
    c, G0, G1 = U
    z = np.zeros_like(c)
    Phi = [[-D * G0 + c * u0, -D * G1 + c * u1, z],
           [G0 * u0 - c / tau_grad, G0 * u1, z],
           [G1 * u0, G1 * u1 - c / tau_grad, z]]
    return Phi


def flux_urf_listing(U):
    """SM4.4, PAPER.md:L849 (ideal ultrarelativistic fluid, expanded component form)."""
    E, S0, S1 = U
    z = np.zeros_like(E)
    root = np.sqrt(4 * E**2 - 3 * S0**2 - 3 * S1**2)
    P10 = -E / 3 + 3 * S0**2 / (2 * E + root) + root / 3
    P11 = 3 * S0 * S1 / (2 * E + root)
    P21 = -E / 3 + 3 * S1**2 / (2 * E + root) + root / 3
    return [[S0, S1, z], [P10, P11, z], [P11, P21, z]]


def flux_maxwell_listing(U, c):
    """SM4.5, PAPER.md:L861 (Maxwell TM)."""
    Ez, Hx, Hy = U
    z = np.zeros_like(Ez)
    return [[-Hy * c, Hx * c, z], [z, Ez * c, z], [-Ez * c, z, z]]


def flux_allencahn_listing(U, gamma, r, tau_grad):
    """SM4.8, PHYSICAL tracker G = grad phi. Returns (Phi, S) physical."""
    phi, G0, G1 = U
    z = np.zeros_like(phi)
    Phi = [[-G0 * gamma, -G1 * gamma, z], [-phi / tau_grad, z, z], [z, -phi / tau_grad, z]]
    S = [-phi**3 * r + phi * r, -G0 / tau_grad, -G1 / tau_grad]
    return Phi, S


def flux_inse_listing(U, cs, mu, tau_grad):
    """SM4.9, PAPER.md:L947-L959 (weakly compressible NSE), PHYSICAL trackers G_ab = d_b (rho u_a); the tracker rows
    follow the vector form G (x) u - I (x) rho u / tau_grad of eq (3.22) (L452) where the listing is garbled (L955).
    U = (rho, ru0, ru1, G00, G01, G10, G11).  Returns (Phi, S) physical."""
    rho, ru0, ru1, G00, G01, G10, G11 = U
    z = np.zeros_like(rho)
    P11 = -G01 * mu / rho - G10 * mu / rho + ru0 * ru1 / rho
    Phi = [[ru0, ru1, z],
           [-2 * G00 * mu / rho + cs**2 * rho + ru0**2 / rho, P11, z],
           [P11, -2 * G11 * mu / rho + cs**2 * rho + ru1**2 / rho, z],
           [G00 * ru0 / rho - ru0 / tau_grad, G00 * ru1 / rho, z],
           [G01 * ru0 / rho, G01 * ru1 / rho - ru0 / tau_grad, z],
           [G10 * ru0 / rho - ru1 / tau_grad, G10 * ru1 / rho, z],
           [G11 * ru0 / rho, G11 * ru1 / rho - ru1 / tau_grad, z]]
    S = [z, z, z, -G00 / tau_grad, -G01 / tau_grad, -G10 / tau_grad, -G11 / tau_grad]
    return Phi, S


def flux_elasticity_listing(U, rho0, mu_s, lambda_s):
    """SM4.6, PAPER.md:L871-L895 (state (F_00, F_01, F_10, F_11, v_0, v_1), shared subexpressions chi_0..chi_8)."""
    F00, F01, F10, F11, v0, v1 = U
    z = np.zeros_like(F00)
    chi0, chi1, chi2 = -v0, -v1, mu_s / rho0
    chi3, chi4 = F00 * F11, F01 * F10
    chi5 = 1 / (chi3 * rho0 - chi4 * rho0)
    chi6 = np.log(chi3 - chi4)
    chi7, chi8 = chi5 * chi6 * lambda_s, chi5 * mu_s
    return [[chi0, z, z], [z, chi0, z], [chi1, z, z], [z, chi1, z],
            [-F00 * chi2 + F11 * chi5 * mu_s - F11 * chi7, -F01 * chi2 + F10 * chi5 * chi6 * lambda_s - F10 * chi8, z],
            [F01 * chi5 * chi6 * lambda_s - F01 * chi8 - F10 * chi2, F00 * chi5 * mu_s - F00 * chi7 - F11 * chi2, z]]


def step(f, dim, omega, F_lat, S_lat):
    """One collide-and-stream step.
    f[k][i] : arrays (nz, ny, nx);  F_lat[k][a], S_lat[k] : lattice flux / source arrays at the
    CURRENT moments (computed by the caller from U = sum_i f).  Returns the new f.
    """
    L = LATTICES[dim]
    m, Q = len(f), len(L["c"])
    new = [[None] * Q for _ in range(m)]
    for k in range(m):
        Uk = sum(f[k][i] for i in range(Q))                                   # eq (2.6)
        for i in range(Q):
            cx, cy, cz = L["c"][i]
            cF = cx * F_lat[k][0] + cy * F_lat[k][1] + cz * F_lat[k][2]
            feq = L["w"][i] * (Uk + cF / L["cs2"])                            # eq (2.7)
            post = f[k][i] - omega[k] * (f[k][i] - feq) + L["w"][i] * S_lat[k]  # eq (2.11)
            # f(x + c_i, t + dt) = post(x): shift the array by +c_i along each axis (z, y, x order)
            new[k][i] = np.roll(post, shift=(cz, cy, cx), axis=(0, 1, 2))
    return new


def moments(f):
    return [sum(fk) for fk in f]


def init_equilibrium(U, F_lat, dim):
    L = LATTICES[dim]
    return [[L["w"][i] * (U[k] + (L["c"][i][0] * F_lat[k][0] + L["c"][i][1] * F_lat[k][1] + L["c"][i][2] * F_lat[k][2]) / L["cs2"])
             for i in range(len(L["c"]))] for k in range(len(U))]
