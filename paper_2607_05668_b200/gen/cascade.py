"""Build-time generator: Split / Cascade / Assemble / Emit of Alg 2.1 on a small declarative spec.

Product-side code.  `gen/mms_codegen.py` emits the manufactured residual; this module derives the AUGMENTED SYSTEM itself:
    declare   the conservation laws d_t Q + div Phi(Q, grad ...) = S  in physical form, gradients written as grad(expr)
              (Listing 1 / Listing 2 of the paper: `grad`, `cgrad`)
    Split     into (Q_k, Phi_k, S_k)                                                         (Alg 2.1 lines 3-11, L234-L243)
    Cascade   while a gradient remains: innermost first; the gradient of a transported field (conserved, or a parent declared
              with `track`) becomes a tracker G with  Phi_G = G (x) u - I V/tau_grad,  S_G = -G/tau_grad  (eq 2.2-2.3);
              the gradient of any other expression is expanded by the chain rule over the transported fields (`cgrad`, L282)
                                                                                             (Alg 2.1 lines 12-19, L244-L265)
    Assemble  the augmented state Q+ = (conserved, trackers), its flux and source            (lines 20-23, L266-L273)
    lattice   F = (dt/dx) Phi, s = dt S, trackers carried as G^L = dx G (exponents (p-1, q), L298)
    Emit      CSE'd straight-line C++ (`csrc/cascade_generated.cuh`), one __host__ __device__ function per system
                                                                                             (lines 24-25, L275-L277)
The hand-written delta-form specialisations of csrc/systems.cuh stay the step kernels' code (they cancel the O(1) backgrounds
analytically for fp32, Appendix B of SURVEY.md); the emitted plain forms are what they are CHECKED against: on the host through
`lbmk_generated_flux` (tests/test_cascade_codegen.py: also against the oracle's independent hand derivation) and on the device
through `lbmk_flux_selfcheck` (every node of a live state).

Run from the repo root:   python -m paper_2607_05668_b200.gen.cascade
"""
from __future__ import annotations

import os
import sys
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import sympy as sp

from .mms_codegen import _Printer

dx, dt, gtau = sp.symbols("dx dt gtau", positive=True)
D_ = sp.Function("D_")          # D_(expr, a): d expr / d x_a, the placeholder the cascade resolves


class Laws:
    """Declarative spec of one system (the subset of the paper's DSL the hot path needs)."""

    def __init__(self, name: str, dim: int, fields: Sequence[str], params: Sequence[str], aux: Sequence[str] = ()):
        self.name, self.dim = name, dim
        self.field_names = list(fields)
        self.V = [sp.Symbol(f, real=True) for f in fields]
        self.par = [sp.Symbol(p, real=True) for p in params]
        self.aux = [sp.Symbol(a, real=True) for a in aux]
        self.flux: List[List[sp.Expr]] = []
        self.source: List[sp.Expr] = []
        self.velocity: List[sp.Expr] = [sp.Integer(0)] * dim      # advecting velocity of the trackers (eq 2.3)
        self.tracked: Dict[sp.Expr, str] = {}                    # derived parents transported directly (`track`)
        self.custom: List[Tuple[str, List[sp.Expr]]] = []        # trackers of a LINEAR COMBINATION of gradients (`track_combination`)

    def grad(self, e) -> List[sp.Expr]:
        return [D_(e, sp.Integer(a)) for a in range(self.dim)]

    def track(self, name: str, e: sp.Expr):
        """Declare a derived parent whose gradient gets its own tracker (eq 3.27's reduced basis tracks u and T directly)."""
        self.tracked[sp.sympify(e)] = name

    def track_combination(self, name: str, injection: Sequence[sp.Expr]) -> sp.Symbol:
        """A tracker of a linear combination of first derivatives, T = sum_j d_j (injection_j): flux T (x) u - injection/tau_grad, source
        -T/tau_grad (eq 2.3 applied to the combination).  HCNSF's reduced basis tracks sym grad u this way (Phi = G_u (x) u -
        sym(I (x) u)/tau_grad); config 5 tracks the current density J = curl B."""
        g = sp.Symbol(f"G_{name}", real=True)
        self.custom.append((g, [sp.sympify(c) for c in injection]))
        return g

    def add(self, flux_rows: Sequence[Sequence[sp.Expr]], sources: Sequence[sp.Expr]):
        assert len(flux_rows) == len(self.V) == len(sources)
        self.flux = [[sp.sympify(c) for c in r] for r in flux_rows]
        self.source = [sp.sympify(c) for c in sources]


class Augmented:
    def __init__(self, laws: Laws, names, Q, Phi, S, parents):
        self.laws, self.names, self.Q, self.Phi, self.S, self.parents = laws, names, Q, Phi, S, parents
        self.m = len(Q)


def cascade(laws: Laws) -> Augmented:
    """Alg 2.1 Split / Cascade / Assemble.  Returns the augmented system in PHYSICAL form (trackers G = grad V)."""
    tau = gtau * dt
    names = list(laws.field_names)
    Q = list(laws.V)
    Phi = [list(r) for r in laws.flux]
    S = list(laws.source)
    parents: List[Optional[Tuple[sp.Expr, int]]] = [None] * len(Q)
    tracker_of: Dict[Tuple[sp.Expr, int], sp.Symbol] = {}
    u = laws.velocity

    def register(parent: sp.Expr, pname: str, a: int) -> sp.Symbol:
        key = (parent, a)
        if key in tracker_of:
            return tracker_of[key]
        g = sp.Symbol(f"G_{pname}_{a}", real=True)
        tracker_of[key] = g
        names.append(str(g)); Q.append(g); parents.append(key)
        Phi.append([g * u[j] - (parent / tau if j == a else 0) for j in range(laws.dim)])    # eq 2.3
        S.append(-g / tau)
        return g

    def resolve(e: sp.Expr) -> sp.Expr:
        # the while-loop of L244-L265: innermost gradient first
        while True:
            atoms = sorted(e.atoms(D_), key=sp.default_sort_key)
            if not atoms:
                return e
            inner = [a for a in atoms if not a.args[0].atoms(D_)]
            a = inner[0]
            arg, ax = a.args[0], int(a.args[1])
            if arg in laws.V or arg in tracker_of.values():
                rep = register(arg, str(arg), ax)
            elif arg in laws.tracked:
                rep = register(arg, laws.tracked[arg], ax)
            else:                                       # chain rule over the transported fields (cgrad, L282)
                rep = sum(sp.diff(arg, v) * D_(v, sp.Integer(ax)) for v in laws.V + list(tracker_of.values()) if arg.has(v))
            e = e.xreplace({a: rep})

    for g, inj in laws.custom:                          # declared combination trackers (their symbols already appear in the fluxes)
        names.append(str(g)); Q.append(g); parents.append((g, -1))
        Phi.append([g * u[j] - inj[j] / tau for j in range(laws.dim)])
        S.append(-g / tau)
    k = 0
    while k < len(Q):                                   # rows appended by register() are resolved too (nested cascades)
        Phi[k] = [resolve(sp.sympify(c)) for c in Phi[k]]
        S[k] = resolve(sp.sympify(S[k]))
        k += 1
    return Augmented(laws, names, Q, Phi, S, parents)


def to_lattice(aug: Augmented):
    """F = (dt/dx) Phi, s = dt S, trackers in lattice units G^L = dx G (rows of trackers scaled by dx, symbols substituted)."""
    il = dt / dx
    sub = {q: q / dx for q, p in zip(aug.Q, aug.parents) if p is not None}
    F, s = [], []
    for k in range(aug.m):
        scale = dx if aug.parents[k] is not None else 1
        F.append([sp.together(sp.expand(scale * il * c.xreplace(sub))) for c in aug.Phi[k]])
        s.append(sp.together(sp.expand(scale * dt * aug.S[k].xreplace(sub))))
    return F, s


# ------------------------------------------------------------------------------------------------ the systems
def euler2d():
    L = Laws("euler2d", 2, ["rho", "m0", "m1", "E"], ["gamma"])
    rho, m0, m1, E = L.V
    g, = L.par
    u = [m0 / rho, m1 / rho]
    p = (g - 1) * (E - rho * (u[0]**2 + u[1]**2) / 2)
    L.add([[m0, m1], [m0 * u[0] + p, m0 * u[1]], [m1 * u[0], m1 * u[1] + p], [(E + p) * u[0], (E + p) * u[1]]], [0, 0, 0, 0])   # eq 3.4
    return L


def swe2d_bathy():
    L = Laws("swe2d_bathy", 2, ["h", "q0", "q1"], ["g"], aux=["zb0", "zb1"])
    h, q0, q1 = L.V
    g, = L.par
    u = [q0 / h, q1 / h]
    P = g * h * h / 2
    L.add([[q0, q1], [q0 * u[0] + P, q0 * u[1]], [q1 * u[0], q1 * u[1] + P]], [0, -g * h * L.aux[0], -g * h * L.aux[1]])          # eq 3.6
    return L


def adr2d():
    L = Laws("adr2d", 2, ["c"], ["u0", "u1", "Dc", "Rc"])
    c, = L.V
    u0, u1, Dc, Rc = L.par
    L.velocity = [u0, u1]
    gc = L.grad(c)
    L.add([[u0 * c - Dc * gc[0], u1 * c - Dc * gc[1]]], [Rc * c * (1 - c)])                                                      # eq 3.17
    return L


def allencahn2d():
    L = Laws("allencahn2d", 2, ["phi"], ["gam", "r"])
    phi, = L.V
    gam, r = L.par
    gp = L.grad(phi)
    L.add([[-gam * gp[0], -gam * gp[1]]], [r * (phi - phi**3)])                                                                  # eq 3.19
    return L


def inse2d():
    L = Laws("inse2d", 2, ["rho", "m0", "m1"], ["cs", "mu"])
    rho, m0, m1 = L.V
    cs, mu = L.par
    m = [m0, m1]
    u = [m0 / rho, m1 / rho]
    L.velocity = u
    gm = [L.grad(m0), L.grad(m1)]
    rows = [[m0, m1]]
    for a in range(2):
        rows.append([m[a] * u[j] + (cs**2 * rho if a == j else 0) - mu / rho * (gm[a][j] + gm[j][a]) for j in range(2)])        # eq 3.22
    L.add(rows, [0, 0, 0])
    return L


def _newtonian(L, u, T, mu, K, dim):
    gu = [L.grad(ua) for ua in u]
    gT = L.grad(T)
    div = sum(gu[a][a] for a in range(dim))
    tau = [[mu * (gu[a][b] + gu[b][a]) - (sp.Rational(2, 3) * mu * div if a == b else 0) for b in range(dim)] for a in range(dim)]
    return tau, gT


def nsf2d():
    L = Laws("nsf2d", 2, ["rho", "m0", "m1", "E"], ["gamma", "mu", "K"])
    rho, m0, m1, E = L.V
    g, mu, K = L.par
    m = [m0, m1]
    u = [m0 / rho, m1 / rho]
    L.velocity = u
    p = (g - 1) * (E - rho * (u[0]**2 + u[1]**2) / 2)
    tau, gT = _newtonian(L, u, p / rho, mu, K, 2)                       # gradients of u, T: chain rule over (rho, m, E), L282
    rows = [[m0, m1]]
    for a in range(2):
        rows.append([m[a] * u[j] + (p if a == j else 0) - tau[a][j] for j in range(2)])
    rows.append([(E + p) * u[j] - sum(tau[j][b] * u[b] for b in range(2)) - K * gT[j] for j in range(2)])                       # eq 3.24
    L.add(rows, [0, 0, 0, 0])
    return L


def mhd2d():
    L = Laws("mhd2d", 2, ["rho", "m0", "m1", "E", "B0", "B1"], ["gamma", "mu", "K", "eta"])
    rho, m0, m1, E, B0, B1 = L.V
    g, mu, K, eta = L.par
    m, B = [m0, m1], [B0, B1]
    u = [m0 / rho, m1 / rho]
    L.velocity = u
    B2 = B0**2 + B1**2
    p = (g - 1) * (E - rho * (u[0]**2 + u[1]**2) / 2 - B2 / 2)
    pt = p + B2 / 2
    uB = u[0] * B0 + u[1] * B1
    tau, gT = _newtonian(L, u, p / rho, mu, K, 2)
    gB = [L.grad(B0), L.grad(B1)]
    jz = gB[1][0] - gB[0][1]
    jxB = [-jz * B1, jz * B0]
    divB = gB[0][0] + gB[1][1]
    rows = [[m0, m1]]
    for a in range(2):
        rows.append([m[a] * u[j] - B[a] * B[j] + (pt if a == j else 0) - tau[a][j] for j in range(2)])
    rows.append([(E + pt) * u[j] - B[j] * uB - sum(tau[j][b] * u[b] for b in range(2)) - K * gT[j] + eta * jxB[j] for j in range(2)])
    for i in range(2):
        rows.append([B[i] * u[j] - u[i] * B[j] - eta * gB[i][j] for j in range(2)])                                             # eq 3.25
    L.add(rows, [0, -divB * B0, -divB * B1, -divB * uB, -divB * u[0], -divB * u[1]])                                            # Powell, L484
    return L


def nsf3d():
    L = Laws("nsf3d", 3, ["rho", "m0", "m1", "m2", "E"], ["gamma", "mu", "K"])
    rho, m0, m1, m2, E = L.V
    g, mu, K = L.par
    m = [m0, m1, m2]
    u = [mi / rho for mi in m]
    L.velocity = u
    p = (g - 1) * (E - rho * sum(ui**2 for ui in u) / 2)
    T = p / rho
    for a in range(3):
        L.track(f"u{a}", u[a])                                          # derived parents, as eq 3.27's reduced basis (L495-L497)
    L.track("T", T)
    tau, gT = _newtonian(L, u, T, mu, K, 3)
    rows = [m]
    for a in range(3):
        rows.append([m[a] * u[j] + (p if a == j else 0) - tau[a][j] for j in range(3)])
    rows.append([(E + p) * u[j] - sum(tau[j][b] * u[b] for b in range(3)) - K * gT[j] for j in range(3)])                       # eq 3.23
    L.add(rows, [0] * 5)
    return L


def advection2d():
    L = Laws("advection2d", 2, ["U"], ["ax", "ay"])
    L.add([[L.par[0] * L.V[0], L.par[1] * L.V[0]]], [0])
    return L


def burgers2d():
    L = Laws("burgers2d", 2, ["u"], [])
    u, = L.V
    L.add([[u * u / 2, u * u / 2]], [0])                                                                                       # eq 3.1-3.2
    return L


def swe2d():
    L = Laws("swe2d", 2, ["h", "q0", "q1"], ["g"])
    h, q0, q1 = L.V
    g, = L.par
    P = g * h * h / 2
    L.add([[q0, q1], [q0 * q0 / h + P, q0 * q1 / h], [q1 * q0 / h, q1 * q1 / h + P]], [0, 0, 0])                                  # eq 3.6, flat bed
    return L


def urf2d():
    L = Laws("urf2d", 2, ["E", "S0", "S1"], [])
    E, S0, S1 = L.V
    p = (sp.sqrt(4 * E * E - 3 * (S0 * S0 + S1 * S1)) - E) / 3                                                                    # eq 3.9
    v = [S0 / (E + p), S1 / (E + p)]
    L.add([[S0, S1], [S0 * v[0] + p, S0 * v[1]], [S1 * v[0], S1 * v[1] + p]], [0, 0, 0])                                          # eq 3.8
    return L


def maxwell2d():
    L = Laws("maxwell2d", 2, ["Ez", "Hx", "Hy"], ["c"])
    Ez, Hx, Hy = L.V
    c, = L.par
    L.add([[-c * Hy, c * Hx], [0, c * Ez], [-c * Ez, 0]], [0, 0, 0])                                                              # eq 3.11
    return L


def elasticity2d():
    L = Laws("elasticity2d", 2, ["F00", "F01", "F10", "F11", "m0", "m1"], ["rho0", "mus", "las"])
    F00, F01, F10, F11, m0, m1 = L.V
    rho0, mus, las = L.par
    F = [[F00, F01], [F10, F11]]
    v = [m0 / rho0, m1 / rho0]
    J = F00 * F11 - F01 * F10
    FiT = [[F11 / J, -F10 / J], [-F01 / J, F00 / J]]
    Pk = [[mus * (F[i][j] - FiT[i][j]) + las * sp.log(J) * FiT[i][j] for j in range(2)] for i in range(2)]                        # eq 3.14
    L.add([[-v[0], 0], [0, -v[0]], [-v[1], 0], [0, -v[1]], [-Pk[0][0], -Pk[0][1]], [-Pk[1][0], -Pk[1][1]]], [0] * 6)            # eq 3.15
    return L


def hcnsf3d():
    L = Laws("hcnsf3d", 3, ["rho", "m0", "m1", "m2", "E"], ["gamma", "mu", "kappa", "eta"], aux=["alpha", "us0", "us1", "us2"])
    rho, m0, m1, m2, E = L.V
    g, mu, kappa, eta = L.par
    al, us = L.aux[0], L.aux[1:]
    m = [m0, m1, m2]
    u = [mi / rho for mi in m]
    L.velocity = u
    p = (g - 1) * (E - rho * sum(ui**2 for ui in u) / 2)
    T = p / rho
    L.track("T", T)
    # reduced basis: the SYMMETRIC velocity gradient, six trackers D_ab = (d_b u_a + d_a u_b)/2
    pairs = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    Dsym = {}
    for a, b in pairs:
        inj = [(u[b] if j == a else 0) / 2 + (u[a] if j == b else 0) / 2 for j in range(3)]
        Dsym[(a, b)] = Dsym[(b, a)] = L.track_combination(f"D{a}{b}", inj)
    tr = Dsym[(0, 0)] + Dsym[(1, 1)] + Dsym[(2, 2)]
    tau = [[mu * (2 * Dsym[(a, b)] - (sp.Rational(2, 3) * tr if a == b else 0)) for b in range(3)] for a in range(3)]
    gT = L.grad(T)
    rows = [m]
    for a in range(3):
        rows.append([m[a] * u[j] + (p if a == j else 0) - al * tau[a][j] for j in range(3)])
    rows.append([(E + p) * u[j] - al * sum(tau[j][b] * u[b] for b in range(3)) - al * kappa * gT[j] for j in range(3)])         # eq 3.27
    drag = [(1 - al) / eta * (rho * us[a] - m[a]) for a in range(3)]
    L.add(rows, [0] + drag + [sum(drag[a] * u[a] for a in range(3))])
    return L


def mhd3d():
    L = Laws("mhd3d", 3, ["rho", "m0", "m1", "m2", "E", "B0", "B1", "B2"], ["gamma", "eta"])
    rho, m0, m1, m2, E, B0, B1, B2 = L.V
    g, eta = L.par
    m, B = [m0, m1, m2], [B0, B1, B2]
    u = [mi / rho for mi in m]
    L.velocity = u
    Bsq = sum(b * b for b in B)
    p = (g - 1) * (E - rho * sum(ui**2 for ui in u) / 2 - Bsq / 2)
    pt = p + Bsq / 2
    uB = sum(u[a] * B[a] for a in range(3))
    eps = sp.LeviCivita
    # current density J_i = eps_ijk d_j B_k as a combination tracker: injection_j = eps_ijk B_k (C5)
    Jt = [L.track_combination(f"J{i}", [sum(eps(i, j, k) * B[k] for k in range(3)) for j in range(3)]) for i in range(3)]
    JxB = [Jt[1] * B[2] - Jt[2] * B[1], Jt[2] * B[0] - Jt[0] * B[2], Jt[0] * B[1] - Jt[1] * B[0]]
    rows = [m]
    for a in range(3):
        rows.append([m[a] * u[j] - B[a] * B[j] + (pt if a == j else 0) for j in range(3)])
    rows.append([(E + pt) * u[j] - B[j] * uB + eta * JxB[j] for j in range(3)])
    for i in range(3):
        rows.append([B[i] * u[j] - u[i] * B[j] + eta * sum(eps(i, j, k) * Jt[k] for k in range(3)) for j in range(3)])
    L.add(rows, [0] * 8)
    return L


SYSTEMS: List[Callable[[], Laws]] = [euler2d, swe2d_bathy, adr2d, allencahn2d, inse2d, nsf2d, mhd2d, nsf3d,
                                     advection2d, burgers2d, swe2d, urf2d, maxwell2d, elasticity2d, hcnsf3d, mhd3d]

# order of the augmented components in csrc/systems.cuh / oracle (trackers listed parent by parent, axis fastest)
ORDER = {
    "euler2d": ["rho", "m0", "m1", "E"],
    "swe2d_bathy": ["h", "q0", "q1"],
    "adr2d": ["c", "G_c_0", "G_c_1"],
    "allencahn2d": ["phi", "G_phi_0", "G_phi_1"],
    "inse2d": ["rho", "m0", "m1", "G_m0_0", "G_m0_1", "G_m1_0", "G_m1_1"],
    "nsf2d": ["rho", "m0", "m1", "E"] + [f"G_{v}_{b}" for v in ("rho", "m0", "m1", "E") for b in range(2)],
    "mhd2d": ["rho", "m0", "m1", "E", "B0", "B1"] + [f"G_{v}_{b}" for v in ("rho", "m0", "m1", "E", "B0", "B1") for b in range(2)],
    "nsf3d": ["rho", "m0", "m1", "m2", "E"] + [f"G_u{a}_{b}" for a in range(3) for b in range(3)] + [f"G_T_{b}" for b in range(3)],
    "advection2d": ["U"], "burgers2d": ["u"], "swe2d": ["h", "q0", "q1"], "urf2d": ["E", "S0", "S1"], "maxwell2d": ["Ez", "Hx", "Hy"],
    "elasticity2d": ["F00", "F01", "F10", "F11", "m0", "m1"],
    "hcnsf3d": ["rho", "m0", "m1", "m2", "E", "G_D00", "G_D11", "G_D22", "G_D01", "G_D02", "G_D12", "G_T_0", "G_T_1", "G_T_2"],
    "mhd3d": ["rho", "m0", "m1", "m2", "E", "B0", "B1", "B2", "G_J0", "G_J1", "G_J2"],
}


# ------------------------------------------------------------------------------------------------ assemble in the build's order
def assemble(mk: Callable[[], Laws]):
    """(laws, F[m][dim], s[m]) in lattice form, components permuted into ORDER[name]."""
    laws = mk()
    aug = cascade(laws)
    F, s = to_lattice(aug)
    order = ORDER[laws.name]
    assert sorted(order) == sorted(aug.names), (laws.name, order, aug.names)
    perm = [aug.names.index(n) for n in order]
    # the state symbols of the emitted code are U[k] in the build's order
    Usym = [sp.Symbol(f"U{k}", real=True) for k in range(len(order))]
    sub = {aug.Q[perm[k]]: Usym[k] for k in range(len(order))}
    sub.update({a: sp.Symbol(f"A{i}", real=True) for i, a in enumerate(laws.aux)})
    sub.update({p: sp.Symbol(f"par{i}", real=True) for i, p in enumerate(laws.par)})
    F = [[F[perm[k]][a].xreplace(sub) for a in range(laws.dim)] for k in range(len(order))]
    s = [s[perm[k]].xreplace(sub) for k in range(len(order))]
    return laws, F, s


def numeric(mk: Callable[[], Laws]):
    """lambdify'd (U, A, par, dx, dt, gtau) -> (F[m][dim], s[m]) for tests."""
    laws, F, s = assemble(mk)
    m = len(F)
    args = [sp.Symbol(f"U{k}", real=True) for k in range(m)] + [sp.Symbol(f"A{i}", real=True) for i in range(len(laws.aux))] \
        + [sp.Symbol(f"par{i}", real=True) for i in range(len(laws.par))] + [dx, dt, gtau]
    fn = sp.lambdify(args, [c for r in F for c in r] + s, "math")

    def call(U, A, par, dx_, dt_, gtau_):
        out = fn(*list(U), *list(A)[:len(laws.aux)], *list(par)[:len(laws.par)], dx_, dt_, gtau_)
        import numpy as np
        return np.array(out[:m * laws.dim], dtype=float).reshape(m, laws.dim), np.array(out[m * laws.dim:], dtype=float)
    return laws, call


# ------------------------------------------------------------------------------------------------ emit
HEADER = """// cascade_generated.cuh -- GENERATED by paper_2607_05668_b200/gen/cascade.py; do not edit.
//
// Lattice flux F_k = (dt/dx) Phi_k(Q+) and source s_k = dt S_k(Q+) of the AUGMENTED systems that Alg 2.1 of the paper
// (Split / Cascade / Assemble, PAPER.md:L221-L278) derives from the declared conservation laws: every gradient of a transported
// field is a tracker G^L = dx grad V with flux G u/lambda - I V/g_tau and source -G/g_tau (eq 2.2-2.3), gradients of derived
// quantities are expanded by the chain rule (L282).  Plain (unshifted) forms, CSE'd, one function per system; the step kernels
// use the hand-written delta forms of systems.cuh and are CHECKED against these (lbmk_generated_flux, lbmk_flux_selfcheck).
#pragma once

namespace lbmk {

template <class R> struct GenArgs { R par[8]; R dx, dt, gtau; };

"""


def emit(mk: Callable[[], Laws]) -> str:
    laws, F, s = assemble(mk)
    m, D = len(F), laws.dim
    pr = _Printer("R")
    exprs = [c for r in F for c in r] + s
    repl, red = sp.cse(exprs, symbols=sp.numbered_symbols("v"), optimizations="basic")
    free = set()
    for _, e in repl:
        free |= e.free_symbols
    for e in red:
        free |= e.free_symbols
    free -= {v for v, _ in repl}
    o = [f"// ---- {laws.name}: m = {m} ({len(laws.V)} conserved + {m - len(laws.V)} trackers), dim = {D}, {len(laws.aux)} prescribed fields",
         f"struct Gen_{laws.name} {{",
         f"    static constexpr int M = {m}, D = {D}, NA = {len(laws.aux)};",
         "    template <class R>",
         "    static __host__ __device__ inline void flux(const R* U, const R* A, const GenArgs<R>& a, R* F, R* S) {",
         "        (void)U; (void)A; (void)a;"]
    for sym in sorted(free, key=str):
        n = str(sym)
        if n in ("dx", "dt", "gtau"):
            o.append(f"        const R {n} = a.{n};")
        elif n.startswith("par"):
            o.append(f"        const R {n} = a.par[{int(n[3:])}];")
        elif n[0] == "U":
            o.append(f"        const R {n} = U[{int(n[1:])}];")
        elif n[0] == "A":
            o.append(f"        const R {n} = A[{int(n[1:])}];")
        else:
            raise ValueError(f"unbound symbol {n}")
    for v, e in repl:
        o.append(f"        const R {v} = {pr.doprint(e)};")
    for k in range(m):
        for a in range(D):
            o.append(f"        F[{k * D + a}] = {pr.doprint(red[k * D + a])};")
    for k in range(m):
        o.append(f"        S[{k}] = {pr.doprint(red[m * D + k])};")
    o += ["    }", "};", ""]
    return "\n".join(o)


def generate_text() -> str:
    return HEADER + "\n".join(emit(mk) for mk in SYSTEMS) + "\n}  // namespace lbmk\n"


def main(out_path=None):
    here = os.path.dirname(os.path.abspath(__file__))
    out_path = out_path or os.path.join(os.path.dirname(here), "csrc", "cascade_generated.cuh")
    with open(out_path, "w") as fh:
        fh.write(generate_text())
    print(out_path)


if __name__ == "__main__":
    main(*sys.argv[1:])
