"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself through the same code path: each checks it against
an identity, a closed form, a brute-force re-derivation, or a finite-difference residual.
CPU only (-m "not gpu").
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import OracleGrid

from brute_force import (LATTICES, flux_adr_listing, flux_allencahn_listing, flux_elasticity_listing, flux_euler_listing, flux_inse_listing, flux_maxwell_listing, flux_swe_listing, flux_urf_listing,
                         init_equilibrium, moments, step as bf_step)

SYSTEMS = ["advection2d", "burgers2d", "swe2d", "euler2d", "adr2d", "nsf3d", "mhd3d", "urf2d", "maxwell2d", "allencahn2d", "inse2d", "elasticity2d", "nsf2d"]
PARAMS = {"advection2d": [0.1, 0.05], "burgers2d": [], "swe2d": [1.0], "euler2d": [1.4],
          "adr2d": [0.1, -0.1, 0.01, 1.0], "nsf3d": [1.4, 1e-3, 4.9e-3], "mhd3d": [1.4, 1e-3], "urf2d": [], "maxwell2d": [1.0], "allencahn2d": [0.01, 1.0], "inse2d": [1.0, 0.01], "elasticity2d": [1.3, 1.0, 2.0], "nsf2d": [1.4, 0.0084, 0.0416]}


def small_grid(system, **kw):
    dim = 2 if system.endswith("2d") else 3
    args = dict(system=system, nx=6, ny=5, nz=1 if dim == 2 else 4, dx=1.0 / 16, lam=5.0,
                params=PARAMS[system], tau_R=0.7, g_tau=3.0)
    args.update(kw)
    return OracleGrid(**args)


def physical_state(system, rng, shape=()):
    """A random admissible state (rho, h > 0, p > 0)."""
    m = len(W.COMPONENTS[system])
    U = rng.uniform(-0.3, 0.3, size=(m,) + shape)
    if system in ("swe2d", "euler2d", "nsf3d", "mhd3d", "inse2d", "nsf2d"):
        U[0] = rng.uniform(0.8, 1.2, size=shape)
    if system in ("euler2d", "nsf2d"):
        U[3] = rng.uniform(2.0, 3.0, size=shape)
    if system in ("nsf3d", "mhd3d"):
        U[4] = rng.uniform(2.0, 3.0, size=shape)
    if system in ("advection2d", "burgers2d", "adr2d", "allencahn2d"):
        U[0] = rng.uniform(0.2, 0.9, size=shape)
    if system == "elasticity2d":                # det F > 0: F near the identity
        U[0] = U[0] + 1.0
        U[3] = U[3] + 1.0
    if system == "urf2d":                       # physicality E > |S|
        U[0] = rng.uniform(1.0, 2.0, size=shape)
    return U


# ------------------------------------------------------------------ P1: eq (2.5), (2.8)
@pytest.mark.parametrize("dim", [2, 3])
def test_p1_lattice_isotropy(dim):
    c, w, cs2 = oracle.lattice(dim)
    assert c.shape == (2 * dim + 1, 3)
    assert abs(w.sum() - 1.0) < 1e-15                                   # sum w = 1
    assert np.abs((w[:, None] * c).sum(0)).max() < 1e-15                # sum w c = 0
    M2 = np.einsum("i,ia,ib->ab", w, c, c)                              # sum w c c = cs2 I
    I = np.zeros((3, 3)); I[:dim, :dim] = np.eye(dim)
    assert np.abs(M2 - cs2 * I).max() < 1e-15
    assert cs2 == pytest.approx({2: 1 / 3, 3: 1 / 4}[dim], abs=1e-16)   # Table SM1
    # direction order of SURVEY.md §8(b): 0 rest; 1:+x 2:-x 3:+y 4:-y 5:+z 6:-z
    expect = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)][: 2 * dim + 1]
    assert [tuple(r) for r in c.tolist()] == expect


@pytest.mark.parametrize("system", SYSTEMS)
def test_p1_equilibrium_moments(system):
    """sum_i f_eq = Q_k and sum_i c_i f_eq = (dt/dx) Phi_k exactly (eq 2.8)."""
    g = small_grid(system)
    c, w, cs2 = oracle.lattice(g.dim)
    rng = np.random.default_rng(1)
    for _ in range(5):
        U = rng.normal(size=g.m_total)
        F = rng.normal(size=(g.m_total, 3))
        F[:, g.dim:] = 0.0
        feq = g.equilibrium(U, F)
        assert np.abs(feq.sum(1) - U).max() < 1e-14
        assert np.abs(feq @ c - F).max() < 1e-14
    # and with the system's own flux at an admissible state
    U = physical_state(system, rng)
    F, S = g.flux_source(U)
    feq = g.equilibrium(U, F)
    assert np.abs(feq.sum(1) - U).max() < 1e-14 and np.abs(feq @ c - F).max() < 1e-14
    assert not np.any(F[:, g.dim:])


# ------------------------------------------------------------------ P2: conservation
@pytest.mark.parametrize("system", ["euler2d", "swe2d", "burgers2d", "nsf3d", "mhd3d"])
def test_p2_conserved_totals(system):
    g = small_grid(system, nx=12, ny=10, nz=(1 if system.endswith("2d") else 6), lam=8.0, tau_R=2.0)
    rng = np.random.default_rng(2)
    U = physical_state(system, rng, (g.nz, g.ny, g.nx)) * 1.0
    U[1:] *= 0.2 if system != "burgers2d" else 1.0
    if system in ("euler2d",):
        U[3] = 2.5 + 0.1 * rng.normal(size=U[3].shape)
    if system in ("nsf3d", "mhd3d"):
        U[4] = 2.5 + 0.1 * rng.normal(size=U[4].shape)
    g.init_from_U(U)
    tot0 = g.read_U().reshape(g.m_total, -1).sum(1)
    g.step(40)
    tot1 = g.read_U().reshape(g.m_total, -1).sum(1)
    mc = g.m_conserved
    assert np.abs(tot1[:mc] - tot0[:mc]).max() <= 1e-12 * np.abs(tot0[:mc]).max() * U[0].size ** 0.5


# ------------------------------------------------------------------ P3: Lax-Friedrichs collapse at omega = 1
@pytest.mark.parametrize("system", SYSTEMS)
def test_p3_lax_friedrichs(system):
    """omega = 1 (tau_LB = 1): one step equals the Lax-Friedrichs-type update
       U' = w0 (U+S)(x) + w sum_a [(U+S)(x-e_a) + (U+S)(x+e_a)] - 1/2 sum_a [F_a(x+e_a) - F_a(x-e_a)]."""
    g = small_grid(system, omega=1.0)
    c, w, cs2 = oracle.lattice(g.dim)
    assert w[1] / cs2 == pytest.approx(0.5, abs=1e-16)
    rng = np.random.default_rng(3)
    U = physical_state(system, rng, (g.nz, g.ny, g.nx))
    g.init_from_U(U)
    g.step(1)
    got = g.read_U()
    F = np.zeros((g.m_total, 3) + U.shape[1:]); S = np.zeros_like(U)
    for idx in np.ndindex(U.shape[1:]):
        f_, s_ = g.flux_source(U[(slice(None),) + idx])
        F[(slice(None), slice(None)) + idx] = f_; S[(slice(None),) + idx] = s_
    V = U + S
    exp = w[0] * V
    for a in range(g.dim):
        ax = 3 - a  # array axis of coordinate a in (k, z, y, x)
        exp = exp + w[1] * (np.roll(V, 1, ax) + np.roll(V, -1, ax)) - 0.5 * (np.roll(F[:, a], -1, ax) - np.roll(F[:, a], 1, ax))
    assert np.abs(got - exp).max() < 1e-13


# ------------------------------------------------------------------ P4: config 1 closed forms
def _c1_fourier_exact(U0, a, omega, steps):
    """Exact evolution of the linear scheme per wavevector: F^(t+1) = G(k) F^(t),
       G_ij = exp(-i k.c_i) [(1-omega) delta_ij + omega w_i (1 + c_i.a/cs2)]."""
    L = LATTICES[2]
    c = np.array(L["c"])[:, :2]; w = np.array(L["w"]); cs2 = L["cs2"]
    ny, nx = U0.shape
    Uh = np.fft.fft2(U0)
    ky = 2 * np.pi * np.fft.fftfreq(ny)[:, None]; kx = 2 * np.pi * np.fft.fftfreq(nx)[None, :]
    coef = w * (1.0 + (c @ np.asarray(a)) / cs2)                    # f_eq,i = coef_i U
    out = np.zeros_like(Uh)
    for iy in range(ny):
        for ix in range(nx):
            ph = np.exp(-1j * (kx[0, ix] * c[:, 0] + ky[iy, 0] * c[:, 1]))
            G = ph[:, None] * ((1 - omega) * np.eye(5) + omega * coef[:, None] * np.ones((1, 5)))
            fh = coef * Uh[iy, ix]
            out[iy, ix] = (np.linalg.matrix_power(G, steps) @ fh).sum()
    return np.fft.ifft2(out).real


def test_p4_config1_fourier_exact():
    w = W.c1_advection()
    U0 = w.initial_U()
    got = oracle.run(w)
    tau = 0.5 + w.tau_R * w.dt
    assert tau == pytest.approx(0.8)
    exp = _c1_fourier_exact(U0[0, 0], w.params, 1.0 / tau, w.steps)
    assert np.abs(got[0, 0] - exp).max() < 5e-13


def test_p4_config1_continuous_closed_form():
    """Noise-free field against the translated/decayed solution of the equivalent advection-diffusion
       equation with the relaxation diffusion of eq (2.17)-(2.18), PAPER.md:L186-L190:
       each plane wave moves with a and decays at (tau-1/2) [cs2 |k|^2 - (a.k)^2]."""
    w = W.c1_advection(noise=0.0)
    got = oracle.run(w)[0, 0]
    n, T = w.nx, w.steps
    tau = 0.5 + w.tau_R; ax, ay = w.params; k = 2 * math.pi / n; cs2 = 1 / 3
    y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    xs, ys = x - ax * T, y - ay * T
    # sin sin = 1/2 [cos k(x-y) - cos k(x+y)]
    rm = (tau - 0.5) * (cs2 * 2 * k * k - (ax - ay) ** 2 * k * k)
    rp = (tau - 0.5) * (cs2 * 2 * k * k - (ax + ay) ** 2 * k * k)
    exp = 1.0 + 0.05 * (np.cos(k * (xs - ys)) * math.exp(-rm * T) - np.cos(k * (xs + ys)) * math.exp(-rp * T))
    assert np.abs(got - exp).max() < 2e-4
    # and it is a real test: the undamped translate is far outside the tolerance
    und = 1.0 + 0.1 * np.sin(k * xs) * np.sin(k * ys)
    assert np.abs(got - und).max() > 1e-2


# ------------------------------------------------------------------ P5: omega = 0 is a pure shift, bit-exact
@pytest.mark.parametrize("system,shape", [("euler2d", (1, 5, 7)), ("mhd3d", (3, 4, 5))])
def test_p5_pure_streaming_bit_exact(system, shape):
    nz, ny, nx = shape
    g = small_grid(system, nx=nx, ny=ny, nz=nz, omega=0.0)
    c, _, _ = oracle.lattice(g.dim)
    # integer tags: unique per (k, i, node)
    f0 = np.arange(np.prod(g.shape_f), dtype=np.float64).reshape(g.shape_f)
    g.set_f(f0)
    N = 4
    g.step(N)
    f1 = g.read_f()
    for i in range(g.Q):
        exp = np.roll(f0[:, i], shift=(N * c[i, 2], N * c[i, 1], N * c[i, 0]), axis=(1, 2, 3))
        # tracker components keep their state source -G/g_tau at omega = 0; the pure shift holds for S = 0
        mc = g.m_conserved
        assert np.array_equal(f1[:mc, i], exp[:mc])
    # index map: source node of direction i at x is wrap(x - c_i)
    lin = np.arange(nz * ny * nx, dtype=np.int64).reshape(nz, ny, nx)
    for i in range(g.Q):
        exp = np.roll(lin, shift=(c[i, 2], c[i, 1], c[i, 0]), axis=(0, 1, 2))
        assert np.array_equal(g.stream_index_map(i), exp)


# ------------------------------------------------------------------ P6 / P7: fixed point and the shift identity
@pytest.mark.parametrize("system", ["euler2d", "swe2d", "nsf3d", "mhd3d"])
def test_p6_uniform_state_is_fixed_point(system):
    w = {"euler2d": W.c3_euler(8), "swe2d": W.c2_swe(8), "nsf3d": W.c4_nsf3d(6, mms=False), "mhd3d": W.c5_mhd3d(6)}[system]
    U = np.broadcast_to(np.asarray(w.U_ref)[:, None, None, None], (w.m_total, w.nz, w.ny, w.nx)).copy()
    for shifted in (False, True):
        g = OracleGrid.from_workload(w, shifted=shifted, mms_id=0)
        g.init_from_U(U)
        if shifted:
            assert np.all(g.read_f() == 0.0)
        g.step(7)
        if shifted:
            assert np.all(g.read_f() == 0.0)           # delta = 0 stays exactly 0 (eq 2.23)
        assert np.abs(g.read_U() - U).max() < 1e-14


@pytest.mark.parametrize("name", ["c2", "c3", "c4", "c5"])
def test_p7_shifted_equals_unshifted(name):
    w = {"c2": W.c2_swe(16, steps=20), "c3": W.c3_euler(16, steps=20), "c4": W.c4_nsf3d(8, steps=10),
         "c5": W.c5_mhd3d(8, steps=10)}[name]
    a = oracle.run(w, shifted=False)
    b = oracle.run(w, shifted=True)
    assert np.abs(a - b).max() < 1e-13


# ------------------------------------------------------------------ P9: tracker on a frozen parent
@pytest.mark.parametrize("g_tau,kmode", [(3.0, 1), (6.0, 2)])
def test_p9_tracker_frozen_parent(g_tau, kmode):
    """Steady tracker response to a frozen parent V = cos(kx) (u = 0), derived from the tracker
       collision of SURVEY.md §8(c) A4:  G^/V^ = -beta w (1/D+ - 1/D-) / (1 - alpha[(1-2w)/omega + w(1/D+ + 1/D-)])."""
    nx, ny = 16, 4
    g = OracleGrid("adr2d", nx, ny, 1, dx=1.0 / nx, lam=4.0, params=[0.0, 0.0, 0.0, 0.0], tau_R=1.0, g_tau=g_tau)
    c, w, cs2 = oracle.lattice(2)
    k = 2 * math.pi * kmode / nx
    x = np.arange(nx)[None, None, :] * np.ones((1, ny, 1))
    V = np.cos(k * x)
    U = np.stack([V, 0 * V, 0 * V])
    g.init_from_U(U)
    for _ in range(400):
        g.step(1)
        f = g.read_f()
        f[0] = w[:, None, None, None] * V[None]      # freeze the parent at rest equilibrium
        g.set_f(f)
    G = g.read_U()[1, 0, 0, :]
    omega = 1.0 / (g_tau + 1.0)
    alpha, beta, wn = omega - 1.0 / g_tau, omega / (g_tau * cs2), w[1]
    Dp, Dm = np.exp(1j * k) - 1 + omega, np.exp(-1j * k) - 1 + omega
    ratio = -beta * wn * (1 / Dp - 1 / Dm) / (1 - alpha * ((1 - 2 * wn) / omega + wn * (1 / Dp + 1 / Dm)))
    exp = (ratio * np.exp(1j * k * np.arange(nx))).real
    assert np.abs(G - exp).max() < 1e-12
    # the k -> 0 limit of that response is the lattice gradient i k (eq 2.4), approached at O(k^2)
    def response(kk):
        dp, dm = np.exp(1j * kk) - 1 + omega, np.exp(-1j * kk) - 1 + omega
        return -beta * wn * (1 / dp - 1 / dm) / (1 - alpha * ((1 - 2 * wn) / omega + wn * (1 / dp + 1 / dm)))
    e1, e3 = abs(response(0.01) / 0.01j - 1), abs(response(0.03) / 0.03j - 1)
    assert e1 < 4.0 * g_tau * (g_tau + 0.5) * cs2 * 1e-4 and 8.0 < e3 / e1 < 10.0
    assert np.abs(g.read_U()[2]).max() < 1e-13       # no y-dependence, no y-gradient


# ------------------------------------------------------------------ P10: MMS forcing vs finite-difference residual
MMS_CASES = {
    "burgers2d": lambda: W.pin_burgers(32),
    "euler2d": lambda: W.pin_euler(32),
    "adr2d": lambda: W.pin_adr(32),
    "swe2d": lambda: W.c2_swe(32),
    "nsf3d": lambda: W.c4_nsf3d(16),
    "urf2d": lambda: W.pin_urf(32),
    "maxwell2d": lambda: W.pin_maxwell(32),
    "allencahn2d": lambda: W.pin_allencahn(32),
    "inse2d": lambda: W.pin_inse(32),
    "elasticity2d": lambda: W.pin_elasticity(32),
    "nsf2d": lambda: W.pin_nsf2d(32),
}


@pytest.mark.parametrize("system", list(MMS_CASES))
def test_p10_mms_forcing_matches_fd_residual(system):
    """s_mms = dt d_t Q + dx div F(Q_exact) - S(Q_exact), eq (4.1) in lattice units, against 4th-order
       central differences of the exact VALUES (no jet derivative enters the reference)."""
    w = MMS_CASES[system]()
    g = OracleGrid.from_workload(w)
    rng = np.random.default_rng(10)
    h = 1e-3

    def d(fun, var, p):
        e = np.zeros(4); e[var] = h
        return (-fun(p + 2 * e) + 8 * fun(p + e) - 8 * fun(p - e) + fun(p - 2 * e)) / (12 * h)

    def Qf(p):
        return g.exact_point(*p)

    def Ff(p):
        return g.flux_source(Qf(p))[0]

    for _ in range(6):
        p = np.concatenate([[rng.uniform(0, 1)], rng.uniform(0, 1, 3)])
        if w.dim == 2:
            p[3] = 0.0
        ref = w.dt * d(Qf, 0, p)
        for a in range(w.dim):
            ref = ref + w.dx * d(lambda q: Ff(q)[:, a], 1 + a, p)
        ref = ref - g.flux_source(Qf(p))[1]
        got = g.mms_source(*p)
        scale = np.abs(ref).max() + 1e-30
        assert np.abs(got - ref).max() < 2e-8 * max(scale, w.dt)


@pytest.mark.parametrize("system", list(MMS_CASES))
def test_exact_fields_match_workload_inputs(system):
    """The oracle's exact fields at t = 0 (incl. tracker components = dx * jet gradient) equal the
       independently typed NumPy initial fields of `workloads` (hand-derived gradients there)."""
    w = MMS_CASES[system]()
    g = OracleGrid.from_workload(w)
    a, b = g.exact_U(0.0), w.initial_U()
    assert np.abs(a - b).max() < 1e-13 * max(1.0, np.abs(b).max())


# ------------------------------------------------------------------ P12: sub-characteristic check
def test_p12_subcharacteristic_violation_detected_and_unstable():
    """Lattice wave speed 1 > c_s is inadmissible (eq 2.19-2.20; Maxwell c = f = 1 example)."""
    c, w, cs2 = oracle.lattice(2)
    bad = OracleGrid("advection2d", 32, 8, 1, dx=1.0, lam=1.0, params=[1.0, 0.0], omega=1.9)
    good = OracleGrid("advection2d", 32, 8, 1, dx=1.0, lam=1.0, params=[0.3, 0.0], omega=1.9)
    x = np.arange(32)[None, None, :] * np.ones((1, 8, 1))
    rng = np.random.default_rng(12)
    U = (1 + 0.1 * np.sin(2 * np.pi * x / 32) + 1e-6 * rng.normal(size=x.shape))[None]
    for g in (bad, good):
        g.init_from_U(U)
    assert bad.max_wave_speed()[0] == pytest.approx(1.0) and bad.max_wave_speed()[0] > math.sqrt(cs2)
    assert good.max_wave_speed()[0] == pytest.approx(0.3) and good.max_wave_speed()[0] < math.sqrt(cs2)
    bad.step(200); good.step(200)
    assert np.abs(good.read_U() - 1).max() < 0.11
    assert not np.all(np.isfinite(bad.read_U())) or np.abs(bad.read_U() - 1).max() > 10.0


def test_wave_speed_values():
    """|u_a| + c with c = sqrt(g h), sqrt(gamma p / rho), fast magnetosonic."""
    g = OracleGrid("swe2d", 4, 4, 1, dx=0.25, lam=2.0, params=[9.0])
    U = np.zeros((3, 1, 4, 4)); U[0] = 4.0; U[1] = 4.0 * 0.5; U[2] = -4.0 * 1.5
    g.init_from_U(U)
    ax, iso, dif = g.max_wave_speed()
    assert ax == pytest.approx((1.5 + 6.0) / 2.0) and iso == pytest.approx((math.hypot(0.5, 1.5) + 6.0) / 2.0) and dif == 0.0
    # MHD: field along x only => fast speed along x is max(a, b), across is sqrt(a^2 + b^2)
    g = OracleGrid("mhd3d", 4, 4, 4, dx=0.25, lam=1.0, params=[1.4, 0.0], g_tau=4.0)
    U = np.zeros((11, 4, 4, 4)); rho, p, Bx = 2.0, 0.5, 3.0
    U[0] = rho; U[5] = Bx; U[4] = p / 0.4 + 0.5 * Bx * Bx
    g.init_from_U(U)
    a2, b2 = 1.4 * p / rho, Bx * Bx / rho
    ax, iso, dif = g.max_wave_speed()
    assert ax == pytest.approx(math.sqrt(a2 + b2)) and iso == pytest.approx(math.sqrt(a2 + b2))


# ------------------------------------------------------------------ P13: brute force on tiny grids
def _bf_run(system, w, steps, listing_flux):
    """NumPy brute force with fluxes from the paper's expanded listings."""
    U = list(w.initial_U())
    dim = w.dim
    il = 1.0 / w.lam
    dt = w.dt
    mc = W.N_CONSERVED[system]
    omega = [1.0 / (0.5 + w.tau_R * dt)] * mc + [1.0 / (w.g_tau + 1.0)] * (w.m_total - mc)

    def lat(Uc):
        if system == "adr2d":
            u0, u1, D, R = w.params
            tau_grad = w.g_tau * dt
            Gphys = [Uc[0], Uc[1] / w.dx, Uc[2] / w.dx]
            Phi = flux_adr_listing(Gphys, u0, u1, D, tau_grad)
            # lattice flux = Phi dt/dx; tracker rows carry an extra dx (G^L = dx G)
            F = [[il * Phi[0][a] for a in range(3)]] + [[il * w.dx * Phi[k][a] for a in range(3)] for k in (1, 2)]
            S = [dt * (-R * Uc[0] ** 2 + R * Uc[0]), dt * (-Uc[1] / tau_grad), dt * (-Uc[2] / tau_grad)]
            return F, S
        if system == "elasticity2d":
            rho0, mus, las = w.params
            Phi = flux_elasticity_listing(list(Uc[:4]) + [Uc[4] / rho0, Uc[5] / rho0], rho0, mus, las)
            F = [[il * Phi[k][a] for a in range(3)] for k in range(4)] + [[il * rho0 * Phi[k][a] for a in range(3)] for k in (4, 5)]
            return F, [0.0 * Uc[0] for _ in Uc]
        if system == "inse2d":
            cs, mu = w.params
            tau_grad = w.g_tau * dt
            Phi, Sp = flux_inse_listing(list(Uc[:3]) + [Uc[k] / w.dx for k in range(3, 7)], cs, mu, tau_grad)
            F = [[il * Phi[k][a] for a in range(3)] for k in range(3)] + [[il * w.dx * Phi[k][a] for a in range(3)] for k in range(3, 7)]
            return F, [dt * Sp[k] for k in range(3)] + [dt * w.dx * Sp[k] for k in range(3, 7)]
        if system == "allencahn2d":
            gam, r = w.params
            tau_grad = w.g_tau * dt
            Phi, Sp = flux_allencahn_listing([Uc[0], Uc[1] / w.dx, Uc[2] / w.dx], gam, r, tau_grad)
            F = [[il * Phi[0][a] for a in range(3)]] + [[il * w.dx * Phi[k][a] for a in range(3)] for k in (1, 2)]
            return F, [dt * Sp[0], dt * w.dx * Sp[1], dt * w.dx * Sp[2]]
        Phi = listing_flux(Uc)
        return [[il * Phi[k][a] for a in range(3)] for k in range(len(Uc))], [0.0 * Uc[0] for _ in Uc]

    F, S = lat(U)
    f = init_equilibrium(U, F, dim)
    for _ in range(steps):
        Uc = moments(f)
        F, S = lat(Uc)
        f = bf_step(f, dim, omega, F, S)
    return np.stack(moments(f))


def test_p13_brute_force_euler():
    w = W.c3_euler(8, ny=6, steps=12)
    exp = _bf_run("euler2d", w, w.steps, lambda U: flux_euler_listing(U, w.params[0]))
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_p13_brute_force_swe():
    w = W.c2_swe(8, ny=6, steps=12)
    w.mms_id = 0
    exp = _bf_run("swe2d", w, w.steps, lambda U: flux_swe_listing(U, w.params[0]))
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_p13_brute_force_adr_tracker():
    w = W.pin_adr(8)
    w.mms_id = 0
    w.steps = 12
    exp = _bf_run("adr2d", w, w.steps, None)
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_p13_brute_force_allencahn_tracker():
    w = W.pin_allencahn(8)
    w.mms_id = 0
    w.steps = 12
    exp = _bf_run("allencahn2d", w, w.steps, None)
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_p13_brute_force_inse_trackers():
    w = W.pin_inse(8)
    w.mms_id = 0
    w.steps = 12
    exp = _bf_run("inse2d", w, w.steps, None)
    assert np.abs(oracle.run(w) - exp).max() < 1e-13


def test_p13_brute_force_elasticity():
    w = W.pin_elasticity(8)
    w.params = [1.3, 1.0, 2.0]                       # rho0 != 1: the listing carries v, the state rho0 v
    w.mms_id = 0
    w.steps = 12
    U0 = w.initial_U(); U0[4:] *= 1.3
    w.init = lambda _w: U0
    exp = _bf_run("elasticity2d", w, w.steps, None)
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_p13_brute_force_ultrarelativistic():
    w = W.pin_urf(8)
    w.mms_id = 0
    w.steps = 12
    exp = _bf_run("urf2d", w, w.steps, flux_urf_listing)
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_p13_brute_force_maxwell():
    w = W.pin_maxwell(8)
    w.mms_id = 0
    w.steps = 12
    U0 = w.initial_U()
    U0[1] = 0.3 * np.roll(U0[0], 2, axis=2); U0[2] = -0.2 * np.roll(U0[0], 1, axis=1)     # non-trivial H
    w.init = lambda _w: U0
    exp = _bf_run("maxwell2d", w, w.steps, lambda U: flux_maxwell_listing(U, w.params[0]))
    assert np.abs(oracle.run(w) - exp).max() < 1e-14


def test_maxwell_wave_equation_dispersion():
    """Eliminating H gives the scalar wave equation d_tt E_z = c^2 lap E_z: an unforced standing TM
    mode oscillates at omega = c |k| (closed form, independent of the scheme), up to the O(dx^2) scheme error."""
    n = 64
    w = W.pin_maxwell(n)
    w.mms_id = 0
    kx, ky = 2 * np.pi, 4 * np.pi
    om = math.hypot(kx, ky)
    T = 2 * np.pi / om                                  # one period
    w.steps = int(round(T / w.dt))
    U = oracle.run(w)
    t = w.steps * w.dt
    x = (np.arange(n) / n)[None, :]; y = (np.arange(n) / n)[:, None]
    Ez = 0.5 * np.sin(kx * x) * np.sin(ky * y) * np.cos(om * t)
    assert np.abs(U[0, 0] - Ez).max() < 2e-2 * 0.5


def test_urf_and_maxwell_wave_speeds():
    """Closed forms: fluid at rest => sound speed 1/sqrt(3); collinear relativistic addition for a
    moving fluid; Maxwell eigenvalues +-c (L393)."""
    g = OracleGrid("urf2d", 4, 4, 1, dx=0.25, lam=1.0, params=[])
    U = np.zeros((3, 1, 4, 4)); U[0] = 2.0
    g.init_from_U(U)
    ax, iso, _ = g.max_wave_speed()
    assert ax == pytest.approx(1 / math.sqrt(3)) and iso == pytest.approx(1 / math.sqrt(3))
    v = 0.5                                              # S = (4/3) Gamma^2 e v, E = (4/3) Gamma^2 e - e/3 with p = e/3
    G2 = 1 / (1 - v * v); e = 1.7
    U[0] = 4 / 3 * G2 * e - e / 3; U[1] = 4 / 3 * G2 * e * v
    g.init_from_U(U)
    ax, iso, _ = g.max_wave_speed()
    cs = 1 / math.sqrt(3)
    assert ax == pytest.approx((v + cs) / (1 + v * cs)) and iso == pytest.approx((v + cs) / (1 + v * cs))
    g = OracleGrid("maxwell2d", 4, 4, 1, dx=0.25, lam=2.0, params=[0.7])
    g.init_from_U(np.ones((3, 1, 4, 4)))
    assert g.max_wave_speed()[:2] == (pytest.approx(0.35), pytest.approx(0.35))


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_p13_brute_force_3d_stepping(name):
    """3D stepping/streaming logic by brute force (flux values taken pointwise from the oracle's flux
       hook; the 3D fluxes themselves are pinned in test_oracle_physics.py)."""
    w = W.c4_nsf3d(4, ny=3, nz=5, steps=6, mms=False) if name == "c4" else W.c5_mhd3d(4, ny=3, nz=5, steps=6)
    g = OracleGrid.from_workload(w)
    omega = g.omega()

    def lat(Uc):
        Ua = np.stack(Uc)
        F = np.zeros((w.m_total, 3) + Ua.shape[1:]); S = np.zeros_like(Ua)
        for idx in np.ndindex(Ua.shape[1:]):
            f_, s_ = g.flux_source(Ua[(slice(None),) + idx])
            F[(slice(None), slice(None)) + idx] = f_; S[(slice(None),) + idx] = s_
        return [[F[k, a] for a in range(3)] for k in range(w.m_total)], [S[k] for k in range(w.m_total)]

    U = list(w.initial_U())
    F, S = lat(U)
    f = init_equilibrium(U, F, 3)
    for _ in range(w.steps):
        F, S = lat(moments(f))
        f = bf_step(f, 3, omega, F, S)
    assert np.abs(oracle.run(w) - np.stack(moments(f))).max() < 1e-14
