"""Build-time generator: manufactured-solution forcing (eq 4.1) -> CUDA/C++ source.

Product-side code (the CUDA path's counterpart of the paper's "Emit" stage, Alg 2.1 lines 24-25,
PAPER.md:L275-L277).  It shares nothing with `oracle/`: the oracle forms the same residual numerically
with forward-mode jets; here the residual of the AUGMENTED system (trackers forced too, reading A5) is
derived symbolically, once, and printed as straight-line code:

    s_k(x, t) = dt d_t Q_k + dx sum_a d_a F_k,a(Q_exact) - S_k(Q_exact)            (lattice units)

Two layers keep the expression small:
  layer 2  the residual written for abstract primitive fields P(t,x,y,z) (rho, u, p, ...): SymPy applies
           the product/chain rules; every Derivative(P, ...) atom becomes a scalar symbol `P_tx` etc.
  layer 1  the closed form of each such atom from the concrete trigonometric fields.  Every sin/cos/exp
           atom depends on ONE of t, x, y, z (after expand_trig), so it is either a per-step "time scalar"
           (host, fp64) or an entry of a per-axis table (host, fp64, one row per node coordinate).
Both layers are CSE'd together.  Output: `csrc/mms_generated.cuh` (device functions + host table code).

Run from the repo root:   python -m paper_2607_05668_b200.gen.mms_codegen
The generated header is committed; `__graft_entry__.build()` does not need SymPy.
"""
from __future__ import annotations

import os
import sys
from typing import Callable, Dict, List, Sequence, Tuple

import sympy as sp
from sympy.printing.c import C99CodePrinter

t, x, y, z = sp.symbols("t x y z", real=True)
COORDS = (t, x, y, z)
CNAME = {t: "t", x: "x", y: "y", z: "z"}
# scaling symbols shared by all systems
dx, dt, il, gtau = sp.symbols("dx dt il gtau", positive=True)   # il = dt/dx = 1/lambda
TWO_PI = sp.Symbol("TWO_PI", positive=True)


def par(i):
    return sp.Symbol(f"par{i}", real=True)


def mp(i):
    return sp.Symbol(f"mp{i}", real=True)


# ------------------------------------------------------------------------------------------------ systems
# Each system: (name, dim, primitive names, concrete primitive fields, augmented state/flux/source builder)
# builder(P: dict name -> expr, D: callable(expr, coord) -> derivative) -> (Q[m], F[m][dim], S[m])

def sys_burgers2d():
    A = mp(0)
    k = TWO_PI
    prim = {"u": A * sp.sin(k * x) * sp.sin(k * y) * sp.cos(t)}          # eq SM5.1

    def build(P, D):
        u = P["u"]
        return [u], [[il * u * u / 2, il * u * u / 2]], [sp.Integer(0)]   # eq 3.1-3.2
    return "burgers2d", 2, prim, build


def sys_swe2d():
    g = par(0)
    Ah, Au, h0 = mp(0), mp(1), mp(2)
    k = TWO_PI
    prim = {"h": h0 + Ah * sp.sin(k * x) * sp.cos(k * y) * sp.cos(t),
            "u": Au * sp.cos(k * x) * sp.sin(k * y) * sp.cos(t),
            "v": Au * sp.sin(k * x) * sp.sin(k * y) * sp.sin(t)}

    def build(P, D):
        h, u, v = P["h"], P["u"], P["v"]
        Pr = g * h * h / 2                                                # eq 3.6, flat bottom
        Q = [h, h * u, h * v]
        F = [[il * h * u, il * h * v],
             [il * (h * u * u + Pr), il * h * u * v],
             [il * h * u * v, il * (h * v * v + Pr)]]
        return Q, F, [sp.Integer(0)] * 3
    return "swe2d", 2, prim, build


def sys_euler2d():
    gamma = par(0)
    k = TWO_PI
    rho0, cs = sp.Integer(1), sp.Integer(1)                              # non-dimensional, reading A9
    p0 = rho0 * cs * cs / gamma
    drho = sp.Rational(3, 10) * rho0 * sp.sin(k * x) * sp.cos(k * y) * sp.cos(t)   # eq SM5.2
    prim = {"rho": rho0 + drho,
            "u": 3 * cs + sp.Rational(3, 10) * cs * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t),
            "v": 3 * cs + sp.Rational(3, 10) * cs * sp.sin(k * x) * sp.sin(k * y) * sp.sin(t),
            "p": p0 + cs * cs * drho + sp.Rational(1, 5) * p0 * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t)}

    def build(P, D):
        rho, u, v, p = P["rho"], P["u"], P["v"], P["p"]
        E = p / (gamma - 1) + rho * (u * u + v * v) / 2
        Q = [rho, rho * u, rho * v, E]
        F = [[il * rho * u, il * rho * v],                                # eq 3.4
             [il * (rho * u * u + p), il * rho * u * v],
             [il * rho * u * v, il * (rho * v * v + p)],
             [il * (E + p) * u, il * (E + p) * v]]
        return Q, F, [sp.Integer(0)] * 4
    return "euler2d", 2, prim, build


def sys_adr2d():
    ux, uy, Dc, R = par(0), par(1), par(2), par(3)
    k = TWO_PI
    prim = {"c": sp.Rational(1, 2) * sp.sin(k * (x - ux * t)) * sp.cos(k * (y - uy * t)) * sp.exp(-t)
            + sp.Rational(1, 2)}                                          # eq SM5.7

    def build(P, D):
        c = P["c"]
        G = [dx * D(c, x), dx * D(c, y)]                                  # lattice-unit trackers, L298
        DL = Dc * dt / dx**2
        Q = [c, G[0], G[1]]
        F = [[ux * il * c - DL * G[0], uy * il * c - DL * G[1]],         # eq 3.17
             [ux * il * G[0] - c / gtau, uy * il * G[0]],
             [ux * il * G[1], uy * il * G[1] - c / gtau]]
        S = [dt * R * c * (1 - c), -G[0] / gtau, -G[1] / gtau]
        return Q, F, S
    return "adr2d", 2, prim, build


def sys_nsf3d():
    gamma, mu, K = par(0), par(1), par(2)
    U0, Ar, rho0, p0 = mp(0), mp(1), mp(2), mp(3)
    k = TWO_PI
    Dt = sp.exp(-3 * (mu / rho0) * k * k * t)
    sx, cx, sy, cy, sz, cz = sp.sin(k * x), sp.cos(k * x), sp.sin(k * y), sp.cos(k * y), sp.sin(k * z), sp.cos(k * z)
    prim = {"rho": rho0 * (1 + Ar * sx * sy * cz * sp.cos(t)),
            "u0": U0 * sx * cy * cz * Dt,
            "u1": -U0 * cx * sy * cz * Dt,
            "u2": U0 / 2 * cx * cy * sz * Dt,
            "p": p0 + (rho0 * U0 * U0 / 16) * (sp.cos(2 * k * x) + sp.cos(2 * k * y)) * (sp.cos(2 * k * z) + 2) * Dt * Dt}

    def build(P, D):
        X = (x, y, z)
        rho, p = P["rho"], P["p"]
        u = [P["u0"], P["u1"], P["u2"]]
        T = p / rho
        E = p / (gamma - 1) + rho * sum(ua * ua for ua in u) / 2
        G = [[dx * D(u[a], X[b]) for b in range(3)] for a in range(3)]    # G_ab = dx d_b u_a
        H = [dx * D(T, X[b]) for b in range(3)]
        muL, KL = mu * dt / dx**2, K * dt / dx**2
        trG = G[0][0] + G[1][1] + G[2][2]
        sig = [[muL * (G[a][b] + G[b][a]) - (sp.Rational(2, 3) * muL * trG if a == b else 0) for b in range(3)]
               for a in range(3)]
        Q = [rho] + [rho * ua for ua in u] + [E] + [G[a][b] for a in range(3) for b in range(3)] + H
        F = [[il * rho * u[j] for j in range(3)]]                         # eq 3.23
        for a in range(3):
            F.append([il * (rho * u[a] * u[j] + (p if a == j else 0)) - sig[a][j] for j in range(3)])
        F.append([il * (E + p) * u[j] - sum(sig[j][b] * u[b] for b in range(3)) - KL * H[j] for j in range(3)])
        for a in range(3):
            for b in range(3):
                F.append([il * G[a][b] * u[j] - (u[a] / gtau if j == b else 0) for j in range(3)])
        for b in range(3):
            F.append([il * H[b] * u[j] - (T / gtau if j == b else 0) for j in range(3)])
        S = [sp.Integer(0)] * 5 + [-G[a][b] / gtau for a in range(3) for b in range(3)] + [-H[b] / gtau for b in range(3)]
        return Q, F, S
    return "nsf3d", 3, prim, build


def sys_urf2d():
    k = TWO_PI
    prim = {"E": sp.Rational(2, 5) * sp.sin(k * x) * sp.sin(k * y) * sp.cos(t) + 3,          # eq SM5.4
            "Sx": sp.Rational(2, 5) * sp.cos(k * x) * sp.cos(k * y) * sp.sin(t) + sp.Rational(6, 5),
            "Sy": sp.Rational(2, 5) * sp.sin(k * x) * sp.sin(k * y) * sp.sin(t) + sp.Rational(6, 5)}

    def build(P, D):
        E, Sx, Sy = P["E"], P["Sx"], P["Sy"]
        p = (sp.sqrt(4 * E * E - 3 * (Sx * Sx + Sy * Sy)) - E) / 3                             # eq 3.9
        vx, vy = Sx / (E + p), Sy / (E + p)
        Q = [E, Sx, Sy]
        F = [[il * Sx, il * Sy],                                                                # eq 3.8
             [il * (Sx * vx + p), il * Sx * vy],
             [il * Sy * vx, il * (Sy * vy + p)]]
        return Q, F, [sp.Integer(0)] * 3
    return "urf2d", 2, prim, build


def sys_maxwell2d():
    c = par(0)
    kx, ky, om, A = TWO_PI, 2 * TWO_PI, 4, sp.Rational(1, 2)                                    # eq SM5.5
    prim = {"Ez": A * sp.sin(kx * x) * sp.sin(ky * y) * sp.cos(om * t),
            "Hx": A * sp.sin(kx * x) * sp.cos(ky * y) * sp.sin(om * t),
            "Hy": -A * (kx / ky) * sp.cos(kx * x) * sp.sin(ky * y) * sp.sin(om * t)}

    def build(P, D):
        Ez, Hx, Hy = P["Ez"], P["Hx"], P["Hy"]
        Q = [Ez, Hx, Hy]
        F = [[-c * il * Hy, c * il * Hx], [sp.Integer(0), c * il * Ez], [-c * il * Ez, sp.Integer(0)]]   # eq 3.11
        return Q, F, [sp.Integer(0)] * 3
    return "maxwell2d", 2, prim, build


def sys_allencahn2d():
    gam, r = par(0), par(1)
    k = TWO_PI
    prim = {"phi": sp.Rational(7, 10) * sp.sin(k * x) * sp.cos(k * y) * sp.cos(t)}            # eq SM5.8

    def build(P, D):
        phi = P["phi"]
        G = [dx * D(phi, x), dx * D(phi, y)]
        gL = gam * dt / dx**2
        Q = [phi, G[0], G[1]]
        F = [[-gL * G[0], -gL * G[1]], [-phi / gtau, sp.Integer(0)], [sp.Integer(0), -phi / gtau]]   # eq 3.19
        S = [dt * r * (phi - phi**3), -G[0] / gtau, -G[1] / gtau]
        return Q, F, S
    return "allencahn2d", 2, prim, build


def sys_inse2d():
    cs, mu = par(0), par(1)
    U0, rho0 = mp(0), mp(1)
    k = TWO_PI
    Dt = sp.exp(-2 * (mu / rho0 / cs) * k * k * t)                                           # eq SM5.9
    p = -rho0 * U0 * U0 / 4 * (sp.cos(2 * k * x) + sp.cos(2 * k * y)) * Dt * Dt
    prim = {"rho": rho0 + p / cs**2,
            "u0": -U0 * sp.cos(k * x) * sp.sin(k * y) * Dt,
            "u1": U0 * sp.sin(k * x) * sp.cos(k * y) * Dt}

    def build(P, D):
        X = (x, y)
        rho, u = P["rho"], [P["u0"], P["u1"]]
        m = [rho * u[0], rho * u[1]]
        G = [[dx * D(m[a], X[b]) for b in range(2)] for a in range(2)]
        muL = mu * dt / dx**2
        Q = [rho, m[0], m[1]] + [G[a][b] for a in range(2) for b in range(2)]
        F = [[il * m[0], il * m[1]]]                                                          # eq 3.22
        for a in range(2):
            F.append([il * (m[a] * u[j] + (cs**2 * rho if a == j else 0)) - muL / rho * (G[a][j] + G[j][a]) for j in range(2)])
        for a in range(2):
            for b in range(2):
                F.append([il * G[a][b] * u[j] - (m[a] / gtau if j == b else 0) for j in range(2)])
        S = [sp.Integer(0)] * 3 + [-G[a][b] / gtau for a in range(2) for b in range(2)]
        return Q, F, S
    return "inse2d", 2, prim, build


def sys_elasticity2d():
    rho0, mus, las = par(0), par(1), par(2)
    k = TWO_PI
    A = sp.Rational(3, 50)                                                                    # eq SM5.6
    w0 = A * (sp.sin(k * x) * sp.sin(k * y) * sp.cos(t) + sp.sin(k * x) * sp.cos(k * y) * sp.sin(t) / 2 + sp.cos(k * (x + y)) * sp.cos(t) / 4)
    w1 = A * (sp.cos(k * x) * sp.cos(k * y) * sp.sin(t) + sp.cos(k * x) * sp.sin(k * y) * sp.cos(t) / 2 + sp.sin(k * (x - y)) * sp.sin(t) / 4)
    prim = {"F00": 1 + sp.diff(w0, x), "F01": sp.diff(w0, y), "F10": sp.diff(w1, x), "F11": 1 + sp.diff(w1, y),
            "v0": sp.diff(w0, t), "v1": sp.diff(w1, t)}

    def build(P, D):
        F = [[P["F00"], P["F01"]], [P["F10"], P["F11"]]]
        v = [P["v0"], P["v1"]]
        J = F[0][0] * F[1][1] - F[0][1] * F[1][0]
        FiT = [[F[1][1] / J, -F[1][0] / J], [-F[0][1] / J, F[0][0] / J]]
        Pk = [[mus * (F[i][j] - FiT[i][j]) + las * sp.log(J) * FiT[i][j] for j in range(2)] for i in range(2)]   # eq 3.14
        Q = [F[0][0], F[0][1], F[1][0], F[1][1], rho0 * v[0], rho0 * v[1]]
        Fl = [[-il * v[0], sp.Integer(0)], [sp.Integer(0), -il * v[0]], [-il * v[1], sp.Integer(0)], [sp.Integer(0), -il * v[1]],
              [-il * Pk[0][0], -il * Pk[0][1]], [-il * Pk[1][0], -il * Pk[1][1]]]                # eq 3.15
        return Q, Fl, [sp.Integer(0)] * 6
    return "elasticity2d", 2, prim, build


def sys_nsf2d():
    gamma, mu, K = par(0), par(1), par(2)
    k = TWO_PI
    p0 = 1 / gamma                                                                            # rho0 = c_s = 1 (reading A9)
    drho = sp.Rational(1, 5) * sp.sin(k * x) * sp.cos(k * y) * sp.cos(t)                       # eq SM5.10
    prim = {"rho": 1 + drho,
            "u0": 3 + sp.Rational(1, 5) * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t),
            "u1": 2 + sp.Rational(3, 20) * sp.sin(k * x) * sp.sin(k * y) * sp.cos(t),
            "p": p0 + drho + sp.Rational(1, 5) * p0 * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t)}

    def build(P, D):
        X = (x, y)
        rho, p = P["rho"], P["p"]
        u = [P["u0"], P["u1"]]
        T = p / rho
        E = p / (gamma - 1) + rho * (u[0]**2 + u[1]**2) / 2
        V = [rho, rho * u[0], rho * u[1], E]
        G = [[dx * D(V[v], X[b]) for b in range(2)] for v in range(4)]
        muL, KL = mu * dt / dx**2, K * dt / dx**2
        # physical gradients of the derived fields are those of the exact fields: dx d_b u_a etc. (chain rule on exact data)
        gu = [[dx * D(u[a], X[b]) for b in range(2)] for a in range(2)]
        gT = [dx * D(T, X[b]) for b in range(2)]
        divu = gu[0][0] + gu[1][1]
        tau = [[muL * (gu[a][b] + gu[b][a]) - (sp.Rational(2, 3) * muL * divu if a == b else 0) for b in range(2)] for a in range(2)]
        Q = V + [G[v][b] for v in range(4) for b in range(2)]
        F = [[il * V[1], il * V[2]]]
        for a in range(2):
            F.append([il * (V[1 + a] * u[j] + (p if a == j else 0)) - tau[a][j] for j in range(2)])
        F.append([il * (E + p) * u[j] - sum(tau[j][b] * u[b] for b in range(2)) - KL * gT[j] for j in range(2)])
        for v in range(4):
            for b in range(2):
                F.append([il * G[v][b] * u[j] - (V[v] / gtau if j == b else 0) for j in range(2)])
        S = [sp.Integer(0)] * 4 + [-G[v][b] / gtau for v in range(4) for b in range(2)]
        return Q, F, S
    return "nsf2d", 2, prim, build


def sys_swe2d_bathy():
    g = par(0)
    h0, Ah, m0, Am, Azb, wt = mp(0), mp(1), mp(2), mp(3), mp(4), mp(5)
    k = TWO_PI
    prim = {"h": h0 + Ah * sp.sin(k * x) * sp.sin(k * y) * sp.cos(wt * t),            # eq SM5.3
            "mx": m0 + Am * sp.cos(k * x) * sp.cos(k * y) * sp.sin(wt * t),
            "my": m0 + Am * sp.sin(k * x) * sp.sin(k * y) * sp.sin(wt * t),
            "zb": Azb * sp.sin(k * x) * sp.cos(k * y)}                                  # static bed

    def build(P, D):
        h, mx, my, zb = P["h"], P["mx"], P["my"], P["zb"]
        u, v = mx / h, my / h
        Pr = g * h * h / 2
        Q = [h, mx, my]
        F = [[il * mx, il * my],                                                        # eq 3.6
             [il * (mx * u + Pr), il * mx * v],
             [il * my * u, il * (my * v + Pr)]]
        S = [sp.Integer(0), -dt * g * h * D(zb, x), -dt * g * h * D(zb, y)]           # bed source -g h grad z_b
        return Q, F, S
    return "swe2d_bathy", 2, prim, build


def sys_mhd2d():
    gamma, mu, K, eta = par(0), par(1), par(2), par(3)
    k = TWO_PI
    p0 = 1 / gamma                                                                            # rho0 = c_s = 1 (reading A9)
    drho = sp.Rational(3, 10) * sp.sin(k * x) * sp.cos(k * y) * sp.cos(t)                      # SM5.12
    prim = {"rho": 1 + drho,
            "u0": 3 + sp.Rational(3, 10) * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t),
            "u1": 3 + sp.Rational(3, 10) * sp.sin(k * x) * sp.sin(k * y) * sp.sin(t),
            "p": p0 + drho + sp.Rational(1, 5) * p0 * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t),
            "B0": sp.Rational(1, 2) - sp.Rational(3, 10) * sp.cos(k * x) * sp.sin(k * y) * sp.sin(t),
            "B1": sp.Rational(1, 2) + sp.Rational(3, 10) * sp.sin(k * x) * sp.cos(k * y) * sp.sin(t)}

    def build(P, D):
        X = (x, y)
        rho, p = P["rho"], P["p"]
        u = [P["u0"], P["u1"]]
        B = [P["B0"], P["B1"]]
        T = p / rho
        B2 = B[0]**2 + B[1]**2
        E = p / (gamma - 1) + rho * (u[0]**2 + u[1]**2) / 2 + B2 / 2
        pt = p + B2 / 2
        uB = u[0] * B[0] + u[1] * B[1]
        V = [rho, rho * u[0], rho * u[1], E, B[0], B[1]]
        G = [[dx * D(V[v], X[b]) for b in range(2)] for v in range(6)]
        muL, KL, etaL = mu * dt / dx**2, K * dt / dx**2, eta * dt / dx**2
        gu = [[dx * D(u[a], X[b]) for b in range(2)] for a in range(2)]
        gT = [dx * D(T, X[b]) for b in range(2)]
        divu = gu[0][0] + gu[1][1]
        tau = [[muL * (gu[a][b] + gu[b][a]) - (sp.Rational(2, 3) * muL * divu if a == b else 0) for b in range(2)] for a in range(2)]
        jz = G[5][0] - G[4][1]
        jxB = [-jz * B[1], jz * B[0]]
        divB = G[4][0] + G[5][1]
        Q = V + [G[v][b] for v in range(6) for b in range(2)]
        F = [[il * V[1], il * V[2]]]                                                          # eq 3.25
        for a in range(2):
            F.append([il * (V[1 + a] * u[j] - B[a] * B[j] + (pt if a == j else 0)) - tau[a][j] for j in range(2)])
        F.append([il * ((E + pt) * u[j] - B[j] * uB) - sum(tau[j][b] * u[b] for b in range(2)) - KL * gT[j] + etaL * jxB[j]
                  for j in range(2)])
        for i in range(2):
            F.append([il * (B[i] * u[j] - u[i] * B[j]) - etaL * G[4 + i][j] for j in range(2)])
        for v in range(6):
            for b in range(2):
                F.append([il * G[v][b] * u[j] - (V[v] / gtau if j == b else 0) for j in range(2)])
        S = [sp.Integer(0), -il * divB * B[0], -il * divB * B[1], -il * divB * uB, -il * divB * u[0], -il * divB * u[1]]
        S += [-G[v][b] / gtau for v in range(6) for b in range(2)]
        return Q, F, S
    return "mhd2d", 2, prim, build


SYSTEMS = [sys_burgers2d, sys_swe2d, sys_euler2d, sys_adr2d, sys_nsf3d, sys_urf2d, sys_maxwell2d, sys_allencahn2d, sys_inse2d,
           sys_elasticity2d, sys_nsf2d, sys_swe2d_bathy, sys_mhd2d]


# ------------------------------------------------------------------------------------------------ printing
class _Printer(C99CodePrinter):
    """C printer with R(...)-typed literals and multiplications instead of pow()."""

    def __init__(self, real="R"):
        super().__init__()
        self.real = real

    def _lit(self, s):
        return f"{self.real}({s})" if self.real else s

    def _print_Float(self, e):
        return self._lit(repr(float(e)))

    def _print_Integer(self, e):
        return self._lit(f"{int(e)}.0")

    def _print_Rational(self, e):
        return self._lit(f"{int(e.p)}.0/{int(e.q)}.0")

    def _print_Pow(self, e):
        b, ex = e.base, e.exp
        if ex.is_Integer and -8 <= int(ex) <= 8 and int(ex) != 0:
            n = abs(int(ex))
            s = "*".join([self.parenthesize(b, 60)] * n)
            if n > 1:
                s = f"({s})"
            return f"({self._lit('1.0')}/{s})" if int(ex) < 0 else s
        if ex.is_Rational and ex.q == 2 and abs(int(ex.p)) <= 9:                # half-integer powers via sqrt
            n = abs(int(ex.p)) // 2
            root = f"sqrt({self._print(b)})"
            s = "*".join([self.parenthesize(b, 60)] * n + [root])
            if n > 0:
                s = f"({s})"
            return f"({self._lit('1.0')}/{s})" if ex.p < 0 else s
        raise ValueError(f"unsupported power {e}")


def _atom_symbol_name(f, wrt: Sequence[sp.Symbol]) -> str:
    return f.func.__name__ + ("_" + "".join(CNAME[c] for c in wrt) if wrt else "")


def _separate(expr):
    """Rewrite sin/cos atoms whose argument mixes coordinates into products of single-coordinate atoms."""
    repl = {}
    for a in sorted(expr.atoms(sp.sin, sp.cos), key=sp.default_sort_key):
        if len(a.free_symbols & set(COORDS)) > 1:
            repl[a] = sp.expand_trig(a.func(sp.expand(a.args[0])))
    return expr.xreplace(repl) if repl else expr


def generate_system(name, dim, prim_concrete, build):
    X = (x, y, z)[:dim]
    prim_concrete = {k: _separate(v) for k, v in prim_concrete.items()}
    # ---- layer 2: residual for abstract primitives
    Pf = {k: sp.Function(k)(t, x, y, z) for k in prim_concrete}
    Q, F, S = build(Pf, lambda e, c: sp.diff(e, c))
    m = len(Q)
    res = []
    for k in range(m):
        r = dt * sp.diff(Q[k], t) + dx * sum(sp.diff(F[k][a], X[a]) for a in range(dim)) - S[k]
        res.append(r.doit())
    # ---- every abstract atom (function value or derivative) -> scalar symbol
    atom_syms: Dict[sp.Basic, sp.Symbol] = {}
    layer1: List[Tuple[sp.Symbol, sp.Expr]] = []

    def atom_to_symbol(a):
        if a in atom_syms:
            return atom_syms[a]
        if isinstance(a, sp.Derivative):
            f = a.expr
            wrt = []
            for v, n in a.variable_count:
                wrt += [v] * int(n)
            wrt.sort(key=COORDS.index)
        else:
            f, wrt = a, []
        s = sp.Symbol(_atom_symbol_name(f, wrt), real=True)
        concrete = prim_concrete[f.func.__name__]
        for v in wrt:
            concrete = sp.diff(concrete, v)
        atom_syms[a] = s
        layer1.append((s, concrete))
        return s

    def lower(e):
        # atoms() is a set: visit it in a canonical order, so that the layer-1 list, the table indices and everything
        # CSE'd after them do not depend on the interpreter's hash seed
        repl = {}
        for a in sorted(e.atoms(sp.Derivative), key=sp.default_sort_key):
            repl[a] = atom_to_symbol(a)
        e = e.xreplace(repl)
        repl = {}
        for a in sorted(e.atoms(sp.core.function.AppliedUndef), key=sp.default_sort_key):
            repl[a] = atom_to_symbol(a)
        return e.xreplace(repl)

    res_l = [lower(r) for r in res]
    Q_l = [lower(q.doit()) for q in Q]
    # light algebra: cancels the tracker 1/g_tau pair and the rho*u/rho quotients, keeps factored products
    res_l = [sp.factor_terms(sp.expand(r)) for r in res_l]
    # ---- layer 1: closed forms; classify trig/exp atoms into time scalars and per-axis table entries
    tabs: Dict[sp.Symbol, List[sp.Expr]] = {c: [] for c in COORDS}
    tab_syms: Dict[sp.Basic, sp.Symbol] = {}

    def table_symbol(a):
        if a in tab_syms:
            return tab_syms[a]
        fs = a.free_symbols & set(COORDS)
        assert len(fs) == 1, f"atom {a} is not separable"
        c = next(iter(fs))
        s = sp.Symbol(f"{CNAME[c].upper()}{len(tabs[c])}", real=True)
        tabs[c].append(a)
        tab_syms[a] = s
        return s

    layer1_l = []
    for s, e in layer1:
        e = sp.expand(e)
        repl = {a: table_symbol(a) for a in sorted(e.atoms(sp.sin, sp.cos, sp.exp), key=str)}
        e = e.xreplace(repl)
        assert not (e.free_symbols & set(COORDS)), f"{s}: bare coordinate left in {e}"
        layer1_l.append((s, sp.factor_terms(e)))
    return dict(name=name, dim=dim, m=m, layer1=layer1_l, res=res_l, Q=Q_l, tabs=tabs)


def _used_symbols(exprs):
    out = set()
    for e in exprs:
        out |= e.free_symbols
    return out


def _emit_body(assign: List[Tuple[sp.Symbol, sp.Expr]], outputs: List[sp.Expr], out_name: str, pr: _Printer, indent="    "):
    """CSE the layer-1 definitions and the outputs together and print the definitions the outputs need,
    in dependency order.  Returns (code lines, operation count, free input symbols)."""
    l1_syms = [s for s, _ in assign]
    exprs = [e for _, e in assign] + list(outputs)
    repl, red = sp.cse(exprs, symbols=sp.numbered_symbols("v"), optimizations="basic")
    defs = list(repl) + [(l1_syms[i], red[i]) for i in range(len(assign))]
    index_of = {s: i for i, (s, _) in enumerate(defs)}
    out_red = red[len(assign):]
    done, ordered = set(), []

    def visit(i):
        if i in done:
            return
        done.add(i)
        for d in sorted(defs[i][1].free_symbols, key=str):
            if d in index_of:
                visit(index_of[d])
        ordered.append(i)

    for e in out_red:
        for d in sorted(e.free_symbols, key=str):
            if d in index_of:
                visit(index_of[d])
    lines, ops, free = [], 0, set()
    for i in ordered:
        s, e = defs[i]
        lines.append(f"{indent}const {pr.real} {s} = {pr.doprint(e)};")
        ops += int(sp.count_ops(e))
        free |= e.free_symbols
    for k, e in enumerate(out_red):
        lines.append(f"{indent}{out_name}[{k}] = {pr.doprint(e)};")
        ops += int(sp.count_ops(e))
        free |= e.free_symbols
    free -= {defs[i][0] for i in ordered}
    return lines, ops, free


# ------------------------------------------------------------------------------------------------ row / node split
# The step kernels run one thread block per x-row segment, so everything that does not depend on x is the
# same for all threads of a block.  Substituting the closed forms and expanding, every forcing component is
#     s_k(x; y, z, t) = sum_j C_kj(y, z, t) * mon_j(X0.., r..)
# a short polynomial in the x-table entries X# and in the reciprocals r of the (x-dependent) fields that the
# residual divides by (rho for NSF: T = p/rho), with coefficients that are per-row constants.  `row_coeffs`
# evaluates the C_kj once per (y, z) row and step (a tiny pre-kernel, in fp64); `source_row` is what is left
# per node: a few monomials and one FMA per term.
def split_rows(g):
    """Polynomial row/node split; for residuals that are not polynomial in the x-atoms (the ultrarelativistic
    fluid's sqrt) the split degenerates to: row coefficients = the row-uniform table atoms Y#, Z#, T# themselves,
    node code = the direct CSE'd residual reading them from the row table."""
    try:
        return _split_rows_poly(g)
    except (sp.PolynomialError, AssertionError):
        return _split_rows_direct(g)


def _split_rows_direct(g):
    d = dict(g["layer1"])
    outs = [e.xreplace(d) for e in g["res"]]              # closed forms inlined; CSE'd as a whole by _emit_source_row
    free = set()
    for e in outs:
        free |= e.free_symbols
    is_x = lambda s_: str(s_)[0] == "X" and str(s_)[1:].isdigit()
    uni = sorted([s_ for s_ in free if not is_x(s_)], key=str)   # Y#, Z#, T# atoms and the scalars (il, dt, par#, ...)
    C = {u: sp.Symbol(f"C{i}", real=True) for i, u in enumerate(uni)}
    return dict(coefs=uni, node_defs=[], outs=[e.xreplace(C) for e in outs], n_terms=0, direct=True)


def _split_rows_poly(g):
    xs = [sp.Symbol(f"X{i}", real=True) for i in range(len(g["tabs"][x]))]
    xset = set(xs)
    l1 = dict(g["layer1"])
    recips: Dict[sp.Symbol, sp.Symbol] = {}

    def neg_pow(a):
        return a.is_Pow and a.exp.is_Integer and a.exp < 0 and a.base in l1 and bool(l1[a.base].free_symbols & xset)

    def to_recip(a):
        if a.base not in recips:
            recips[a.base] = sp.Symbol(f"r_{a.base}", real=True)
        return recips[a.base] ** (-a.exp)

    lowered = []
    for e in g["res"]:
        e = sp.expand(e).replace(neg_pow, to_recip)
        lowered.append(sp.expand(e.xreplace(l1)))
    gens = xs + [recips[b] for b in sorted(recips, key=str)]
    coefs: List[sp.Expr] = []           # distinct per-row coefficient expressions
    index: Dict[sp.Expr, Tuple[int, int]] = {}

    def coef_ref(c):
        """(index, sign) of coefficient expression c in the row table (shared up to sign)."""
        c = sp.factor_terms(c)
        if c in index:
            return index[c]
        if -c in index:
            i, sg = index[-c]
            return i, -sg
        coefs.append(c)
        index[c] = (len(coefs) - 1, 1)
        return index[c]

    def poly_terms(e, gs):
        if e == 0:
            return []
        P = sp.Poly(e, *gs) if gs else None
        if P is None:
            return [((), e)]
        return [(m, c) for m, c in zip(P.monoms(), P.coeffs())]

    C = lambda i: sp.Symbol(f"C{i}", real=True)
    node_defs: List[Tuple[sp.Symbol, sp.Expr]] = []
    for b in sorted(recips, key=str):                       # r_b = 1 / (polynomial in X with row coefficients)
        den = 0
        for m, c in poly_terms(sp.expand(l1[b]), xs):
            i, sg = coef_ref(c)
            den += sg * C(i) * sp.Mul(*[gx ** ex for gx, ex in zip(xs, m)])
        node_defs.append((recips[b], 1 / den))
    outs = []
    n_terms = 0
    for e in lowered:
        acc = 0
        for m, c in poly_terms(e, gens):
            assert not (c.free_symbols & (xset | set(recips.values()))), "coefficient depends on x"
            i, sg = coef_ref(c)
            acc += sg * C(i) * sp.Mul(*[gx ** ex for gx, ex in zip(gens, m)])
            n_terms += 1
        outs.append(acc)
    return dict(coefs=coefs, node_defs=node_defs, outs=outs, n_terms=n_terms)


def _emit_row_coeffs(sr, pr: _Printer, indent="        "):
    """CSE'd straight-line code c[i] = ... for the per-row coefficients."""
    repl, red = sp.cse(sr["coefs"], symbols=sp.numbered_symbols("u"), optimizations="basic")
    lines, ops, free = [], 0, set()
    for s_, e in repl:
        lines.append(f"{indent}const {pr.real} {s_} = {pr.doprint(e)};")
        ops += int(sp.count_ops(e)); free |= e.free_symbols
    for i, e in enumerate(red):
        lines.append(f"{indent}c[{i}] = (RO)({pr.doprint(e)});")
        ops += int(sp.count_ops(e)); free |= e.free_symbols
    free -= {s_ for s_, _ in repl}
    return lines, ops, free


def _emit_source_row(sr, pr: _Printer, indent="        "):
    """Per-node code: coefficient loads in 4-wide chunks right before first use, monomials CSE'd."""
    n_def = len(sr["node_defs"])
    repl, red = sp.cse([e for _, e in sr["node_defs"]] + sr["outs"], symbols=sp.numbered_symbols("m"), optimizations="basic")
    loaded = set()
    lines, ops = [], 0
    names = {}

    def prepare(e):
        for s_ in sorted(e.free_symbols, key=str):
            n = str(s_)
            if n[0] == "C" and n[1:].isdigit():
                i = int(n[1:])
                if i // 4 not in loaded:
                    loaded.add(i // 4)
                    lines.append(f"{indent}const Vec4<R> q{i // 4} = ld4<SH>(c + {4 * (i // 4)});")
                names[s_] = sp.Symbol(f"q{i // 4}.{'xyzw'[i % 4]}", real=True)
        return e.xreplace(names)

    defs = list(repl) + [(sr["node_defs"][i][0], red[i]) for i in range(n_def)]
    index_of = {s_: i for i, (s_, _) in enumerate(defs)}
    done = set()

    def visit(i):                                   # dependency order: r_* are inputs of CSE temps and outputs of others
        if i in done:
            return
        done.add(i)
        for d in sorted(defs[i][1].free_symbols, key=str):
            if d in index_of:
                visit(index_of[d])
        s_, e = defs[i]
        lines.append(f"{indent}const R {s_} = {pr.doprint(prepare(e))};")

    for k, e in enumerate(red[n_def:]):
        for d in sorted(e.free_symbols, key=str):
            if d in index_of:
                visit(index_of[d])
        lines.append(f"{indent}s[{k}] = {pr.doprint(prepare(e))};")
        ops += int(sp.count_ops(e))
    ops += sum(int(sp.count_ops(defs[i][1])) for i in done)
    return lines, ops


# ------------------------------------------------------------------------------------------------ emission
SCALARS = {"dx": "a.dx", "dt": "a.dt", "il": "a.il", "gtau": "a.gtau", "TWO_PI": "R(6.283185307179586477)"}


def _bind_inputs(free, real, tab_prefix=True):
    """Declarations binding the free symbols of a body to the argument struct / table rows."""
    out = []
    for s in sorted(free, key=str):
        n = str(s)
        if n in SCALARS:
            out.append(f"    const {real} {n} = {SCALARS[n]};")
        elif n.startswith("par"):
            out.append(f"    const {real} {n} = a.par[{int(n[3:])}];")
        elif n.startswith("mp"):
            out.append(f"    const {real} {n} = a.mp[{int(n[2:])}];")
        elif n[0] in "TXYZ" and n[1:].isdigit():
            out.append(f"    const {real} {n} = {n[0]}[{int(n[1:])}];")
        else:
            raise ValueError(f"unbound symbol {n}")
    return out


def _host_expr(e, coord):
    """C++ (double) text of a table atom as a function of the scalar `c` (the coordinate or the time)."""
    pr = _Printer(real="")
    pr._lit = lambda s: s
    e = e.xreplace({coord: sp.Symbol("c"), TWO_PI: sp.Symbol("6.283185307179586477")})
    return pr.doprint(e)


def emit_system(g) -> str:
    name, m, dim = g["name"], g["m"], g["dim"]
    pr = _Printer("R")
    src_lines, src_ops, src_free = _emit_body(g["layer1"], g["res"], "s", pr)
    q_lines, q_ops, q_free = _emit_body(g["layer1"], g["Q"], "q", pr)
    nt, nx_, ny_, nz_ = (len(g["tabs"][c]) for c in COORDS)
    o = []
    o.append(f"// ---- {name}: m = {m}, dim = {dim}; forcing {src_ops} ops, exact state {q_ops} ops")
    o.append(f"struct Mms_{name} {{")
    o.append(f"    static constexpr int M = {m}, NT = {nt}, NX = {nx_}, NY = {ny_}, NZ = {max(nz_, 0)};")
    sr = split_rows(g)
    nc = len(sr["coefs"])
    ncp = (nc + 3) // 4 * 4
    prd = _Printer("R")
    rc_lines, rc_ops, rc_free = _emit_row_coeffs(sr, prd)
    sn_lines, sn_ops = _emit_source_row(sr, pr)
    o.append(f"    // row/node split of the forcing: {nc} per-row coefficients ({rc_ops} ops per row), {sr['n_terms']} terms, {sn_ops} ops per node")
    o.append(f"    static constexpr int NC = {ncp};")
    # host: time scalars and axis rows
    o.append("    // host side (fp64): per-step time scalars and per-axis table rows")
    o.append("    static __host__ __device__ inline void time_scalars(double c, const MmsHostArgs& a, double* T) {")
    o.append("        (void)c; (void)a; (void)T;")
    for i, e in enumerate(g["tabs"][t]):
        o.append(f"        T[{i}] = {_host_bind(_host_expr(e, t))};")
    o.append("    }")
    o.append("    static __host__ __device__ inline void axis_row(int axis, double c, const MmsHostArgs& a, double* row) {")
    o.append("        (void)c; (void)a; (void)row;")
    for ax, cs in enumerate((x, y, z)):
        if not g["tabs"][cs]:
            continue
        o.append(f"        if (axis == {ax}) {{")
        for i, e in enumerate(g["tabs"][cs]):
            o.append(f"            row[{i}] = {_host_bind(_host_expr(e, cs))};")
        o.append("        }")
    o.append("    }")
    # device: forcing and exact state
    for fn, lines, free, outn in (("source", src_lines, src_free, "s"), ("exact", q_lines, q_free, "q")):
        o.append("    template <class R>")
        o.append(f"    static __host__ __device__ __forceinline__ void {fn}(const MmsArgs<R>& a, const R* T, const R* X, const R* Y, const R* Z, R* {outn}) {{")
        o.append("        (void)a; (void)T; (void)X; (void)Y; (void)Z;")
        o += ["    " + l for l in _bind_inputs(free, "R")]
        o += ["    " + l for l in lines]
        o.append("    }")
    # row / node split
    o.append("    // per-row coefficients C(y, z, t) of the forcing polynomial in the x-table entries (see gen/mms_codegen.py split_rows)")
    o.append("    template <class R, class RO>")
    o.append("    static __host__ __device__ __forceinline__ void row_coeffs(const MmsArgs<R>& a, const R* T, const R* Y, const R* Z, RO* c) {")
    o.append("        (void)a; (void)T; (void)Y; (void)Z;")
    o += ["    " + l for l in _bind_inputs(rc_free, "R")]
    o += rc_lines
    for i in range(nc, ncp):
        o.append(f"        c[{i}] = (RO)0;")
    o.append("    }")
    o.append("    // per-node remainder: s_k = sum_j C_kj * monomial_j(X, 1/rho..); c = this row's coefficients (32-byte aligned)")
    o.append("    template <class R, bool SH>")
    o.append("    static __device__ __forceinline__ void source_row(const R* __restrict__ c, const R* X, R* s) {")
    o.append("        (void)c; (void)X;")
    for i in range(nx_):
        o.append(f"        const R X{i} = X[{i}];")
    o += sn_lines
    o.append("    }")
    o.append("};")
    return "\n".join(o)


def _host_bind(text: str) -> str:
    """par<i>/mp<i> symbols inside a host table expression -> a.par[i] / a.mp[i]."""
    import re
    text = re.sub(r"\bpar(\d+)\b", r"a.par[\1]", text)
    text = re.sub(r"\bmp(\d+)\b", r"a.mp[\1]", text)
    return text


HEADER = """// mms_generated.cuh -- GENERATED by paper_2607_05668_b200/gen/mms_codegen.py; do not edit.
//
// Manufactured-solution forcing s_k = dt d_t Q_k + dx div F_k(Q_exact) - S_k(Q_exact) of eq (4.1)
// (PAPER.md:L499-L504) for the AUGMENTED system (trackers forced too), and the exact augmented state
// Q_exact, as straight-line code over per-step time scalars T[] and per-axis table rows X[], Y[], Z[]
// (every trigonometric/exponential atom of the exact fields depends on one coordinate only).
// Exact fields: Burgers eq SM5.1 (L1161), Euler eq SM5.2 (L1175-L1186), ADR eq SM5.7 (L1292); SWE and
// NSF3D are the BASELINE.json configs[1] / configs[3] fields (DESIGN.md "Input recipe").
#pragma once
#include <cmath>

namespace lbmk {

struct MmsHostArgs { double par[16]; double mp[16]; double dx, dt, il, gtau; };
template <class R> struct MmsArgs { R par[8]; R mp[8]; R dx, dt, il, gtau; };

// four consecutive row coefficients, loaded with 128-bit read-only loads (all threads of a block read the same row)
template <class R> struct Vec4 { R x, y, z, w; };
#ifdef __CUDACC__
// SH: p points into shared memory (plain vector load -> LDS.128); otherwise read-only global load
template <bool SH> __device__ __forceinline__ Vec4<float> ld4(const float* p) {
    const float4 v = SH ? *reinterpret_cast<const float4*>(p) : __ldg(reinterpret_cast<const float4*>(p));
    return Vec4<float>{v.x, v.y, v.z, v.w};
}
template <bool SH> __device__ __forceinline__ Vec4<double> ld4(const double* p) {
    const double2* q = reinterpret_cast<const double2*>(p);
    const double2 a = SH ? q[0] : __ldg(q), b = SH ? q[1] : __ldg(q + 1);
    return Vec4<double>{a.x, a.y, b.x, b.y};
}
#endif

"""


def _generate_one(i: int) -> str:
    name, dim, prim, build = SYSTEMS[i]()
    text = emit_system(generate_system(name, dim, prim, build))
    print(f"generated {name}", file=sys.stderr)
    return text


def generate_text(jobs: int = 0) -> str:
    """The whole header as one string.  Systems are generated independently (one process each when jobs != 1) and joined
    in the fixed order of SYSTEMS; nothing in the pipeline depends on set / hash order (atoms are visited in
    sp.default_sort_key order), so the text is a pure function of this file -- tests/test_codegen.py regenerates it
    under a different PYTHONHASHSEED and compares it byte for byte with the tracked csrc/mms_generated.cuh."""
    idx = list(range(len(SYSTEMS)))
    if jobs == 1:
        texts = [_generate_one(i) for i in idx]
    else:
        import multiprocessing as mpx
        with mpx.get_context("spawn").Pool(jobs or min(len(idx), os.cpu_count() or 1)) as pool:
            texts = pool.map(_generate_one, idx, chunksize=1)
    parts = [HEADER]
    for tx in texts:
        parts.append(tx)
        parts.append("")
    parts.append("}  // namespace lbmk\n")
    return "\n".join(parts)


def main(out_path=None):
    here = os.path.dirname(os.path.abspath(__file__))
    out_path = out_path or os.path.join(os.path.dirname(here), "csrc", "mms_generated.cuh")
    text = generate_text()
    with open(out_path, "w") as fh:
        fh.write(text)
    print(out_path)


if __name__ == "__main__":
    main(*sys.argv[1:])
