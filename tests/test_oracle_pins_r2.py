"""Round-2 pins of the oracle terms that had none (VERDICT r1 "What's weak" 2).  CPU only.  None of these re-types an
oracle formula: each compares the oracle's TIME STEPPING (or its flux through a numerical Jacobian) with a textbook closed form.

  P17  NSF3D entropy (thermal) mode at constant pressure decays at kappa k^2, kappa = K (gamma-1)/(gamma rho0)
       (c_p = gamma/(gamma-1), R = 1; eq 3.23): pins the -K_L H term of the energy flux and the
       grad T tracker (injection -T/g_tau, T = p/rho).
  P18  NSF3D standing sound wave: classical attenuation Gamma = k^2/2 [4/3 nu + (gamma-1) kappa]: pins the -2/3 tr G
       coefficient (without it the viscous part would be 2 nu, not 4/3 nu) and the heat flux in the acoustic mode.
  P19  MHD3D resistive decay of B_y = A sin kx at eta k^2 (eq 3.25): pins eta_L eps J in the
       induction flux and the J tracker; Ohmic heating eta |J|^2 appears as entropy where the CURRENT is (cos^2 kx), which
       pins the Poynting term eta_L J x B of the energy flux (without it the heat would appear where the FIELD is, sin^2 kx).
  P20  wave_speeds(): the hyperbolic speeds equal the spectral radius of the numerical Jacobian of the oracle's own flux
       (|u.n| + c for Euler / NSF / weakly compressible NSE / SWE over a bed / MHD 2D fast speed); the tracker-parent
       signal speed out[2] equals the spectral radius of the augmented Jacobian for the purely diffusive pairs, and the sum
       used by the check bounds the spectral radius of the full augmented Jacobian.
  P21  configs[2] (Euler free evolution): the same workload recipe at amplitude 1e-6 against the closed-form LINEAR acoustics of its
       own seeded fields (standing pressure waves, steady entropy part), second-order approach under refinement.
  P22  dynamics of the systems added in round 2: chain-rule viscous shear decay nu k^2 and thermal-mode decay kappa k^2 of NSF 2D (the
       paper's running example) and MHD 2D; MHD 2D resistive decay eta k^2; HCNSF drag towards the solid velocity (exact
       discrete closed form) and porosity-scaled viscous decay alpha nu k^2 (the halves of the symmetric tracker).
  P11  on the configs themselves: c2 at N = 64, 128, 256 and the fp64 build of c4 at N = 16, 32, 64, to a fixed time:
       L2 slope in the paper's band 1.7-2.5.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W

K2PI = 2.0 * np.pi


def _nsf_state(n, rho, ux, p, gamma, dx, H_x=None, G_xx=None):
    """17-component NSF3D state on an (n, 2, 2) grid varying in x only."""
    U = np.zeros((17, 2, 2, n))
    one = np.ones((2, 2, 1))
    U[0] = rho * one
    U[1] = rho * ux * one
    U[4] = (p / (gamma - 1.0) + 0.5 * rho * ux * ux) * one
    if G_xx is not None:
        U[5] = dx * G_xx * one
    if H_x is not None:
        U[14] = dx * H_x * one
    return U


def _nsf_workload(n, mu, K):
    w = W.c4_nsf3d(n, ny=2, nz=2, precision="f64", mms=False, steps=0)
    w.params = [1.4, mu, K]
    return w


def _entropy_amplitude(U, x, gamma):
    """sin(kx) amplitude of s = ln(gamma p) - gamma ln(rho).  Sound waves are isentropic to first order, so the acoustic
    transient the isobaric start excites (the thermal eigenmode carries an O(kappa k/c) velocity) does not contaminate it."""
    rho = U[0, 0, 0]
    u = U[1, 0, 0] / rho
    p = (gamma - 1.0) * (U[4, 0, 0] - 0.5 * rho * u * u)
    s = np.log(gamma * p) - gamma * np.log(rho)
    return 2.0 * np.abs((s * np.sin(K2PI * x)).mean())


def test_p17_nsf3d_thermal_mode_decays_at_kappa_k2():
    n, eps, gamma = 128, 1e-3, 1.4
    rates = []
    for K in (0.0, 2e-2):
        w = _nsf_workload(n, 0.0, K)
        x = np.arange(n) * w.dx
        p0 = 1.0 / gamma
        rho = 1.0 - eps * np.sin(K2PI * x)                       # isobaric: T = p0/rho = T0 (1 + eps sin kx + O(eps^2))
        dT = p0 * eps * K2PI * np.cos(K2PI * x) / rho ** 2        # the tracker's start value d_x T
        U = _nsf_state(n, rho, 0.0 * x, p0 + 0.0 * x, gamma, w.dx, H_x=dT)
        g = oracle.OracleGrid.from_workload(w)
        g.init_from_U(U)
        s1, s2 = int(round(0.4 / w.dt)), int(round(1.6 / w.dt))
        g.step(s1)
        a1 = _entropy_amplitude(g.read_U(), x, gamma)
        g.step(s2 - s1)
        a2 = _entropy_amplitude(g.read_U(), x, gamma)
        g.close()
        rates.append(math.log(a1 / a2) / ((s2 - s1) * w.dt))
    kappa = 2e-2 * (gamma - 1.0) / gamma
    # measured/closed form: 0.905 at N = 64, 0.975 at 128, 0.994 at 256 -- the tracker's O(dx^2) resolution error (L196)
    assert rates[1] - rates[0] == pytest.approx(kappa * K2PI ** 2, rel=0.04)


def _acoustic_energy(U, gamma):
    rho, u = U[0], U[1] / U[0]
    p = (gamma - 1.0) * (U[4] - 0.5 * rho * u * u)
    c2 = 1.0                                                     # gamma p0 / rho0
    return float((0.5 * u * u + 0.5 * (p - 1.0 / gamma) ** 2 / c2).mean())


@pytest.mark.parametrize("mu,K", [(5e-3, 0.0), (0.0, 2e-2)])
def test_p18_nsf3d_sound_attenuation(mu, K):
    n, A, gamma = 128, 1e-4, 1.4
    decay = []
    for (m_, K_) in ((0.0, 0.0), (mu, K)):
        w = _nsf_workload(n, m_, K_)
        x = np.arange(n) * w.dx
        ux = A * np.sin(K2PI * x)
        U = _nsf_state(n, 1.0 + 0.0 * x, ux, 1.0 / gamma + 0.0 * x, gamma, w.dx, G_xx=A * K2PI * np.cos(K2PI * x))
        steps = int(round(2.0 / w.dt))                            # two acoustic periods (c = 1, wavelength 1)
        U1 = oracle.run(w, steps=steps, U0=U)
        decay.append(-math.log(_acoustic_energy(U1, gamma) / _acoustic_energy(U, gamma)) / (2.0 * steps * w.dt))
    kappa = K * (gamma - 1.0) / gamma
    want = 0.5 * K2PI ** 2 * (4.0 / 3.0 * mu + (gamma - 1.0) * kappa)
    assert decay[1] - decay[0] == pytest.approx(want, rel=0.06)
    # the same wave with the bulk coefficient missing (sigma = mu (G + G^T)) would be damped at k^2 nu, 50 % more
    if mu > 0:
        assert abs(decay[1] - decay[0] - 0.5 * K2PI ** 2 * 2.0 * mu) > 0.25 * want


def test_p19_mhd3d_resistive_decay_and_ohmic_heating():
    n, A, gamma, eta = 128, 1e-2, 1.4, 5e-3
    out = []
    for e_ in (0.0, eta):
        w = W.c5_mhd3d(n, ny=2, nz=2, precision="f64", steps=0)
        w.params = [gamma, e_]
        x = np.arange(n) * w.dx
        one = np.ones((2, 2, 1))
        U = np.zeros((11, 2, 2, n))
        By = A * np.sin(K2PI * x)
        U[0] = 1.0
        U[6] = By * one
        U[4] = ((1.0 / gamma) / (gamma - 1.0) + 0.5 * By * By) * one
        U[10] = w.dx * A * K2PI * np.cos(K2PI * x) * one            # J_z = d_x B_y
        steps = int(round(0.25 / w.dt))
        U1 = oracle.run(w, steps=steps, U0=U)
        t = steps * w.dt
        amp = 2.0 * np.abs((U1[6, 0, 0] * np.sin(K2PI * x)).mean())
        rho, m2 = U1[0, 0, 0], (U1[1:4, 0, 0] ** 2).sum(0)
        B2 = (U1[5:8, 0, 0] ** 2).sum(0)
        p = (gamma - 1.0) * (U1[4, 0, 0] - 0.5 * m2 / rho - 0.5 * B2)
        s = np.log(p * gamma) - gamma * np.log(rho)                 # entropy perturbation (c_v units)
        out.append((-math.log(amp / A) / t, 2.0 * (s * np.cos(2 * K2PI * x)).mean(), t, float(U1[4].sum() - U[4].sum())))
        assert abs(out[-1][3]) < 1e-10 * U[4].sum()                 # total energy conserved (flux form)
    assert out[1][0] - out[0][0] == pytest.approx(eta * K2PI ** 2, rel=0.05)
    # Ohmic heating eta J^2 = eta k^2 A^2 (1 + cos 2kx)/2 e^{-2 eta k^2 t}: ds/dt = (gamma-1) eta J^2 / p0, so the cos 2kx
    # entropy amplitude after time t is + (gamma-1) gamma eta k^2 A^2 (1 - e^{-2 eta k^2 t}) / (4 eta k^2); with the
    # Poynting term dropped the heat would sit where B is and the sign of this amplitude would flip
    r = eta * K2PI ** 2
    want = (gamma - 1.0) * gamma * A * A * (1.0 - math.exp(-2.0 * r * out[1][2])) / 4.0
    got = out[1][1] - out[0][1]
    # got/want: 0.93 (t = 0.1), 0.87 (t = 0.25), 0.64 (t = 1) at N = 128 and 0.97 (t = 0.25) at N = 256: the scheme's relaxation
    # diffusion (rate 0.097 for the k mode at N = 128, four times that for this 2k mode) smooths the deposited heat
    assert 0.80 * want <= got <= 1.02 * want


# ------------------------------------------------------------------------------------------------ P20 wave speeds
def _jacobian(o, U, A, axis, h=1e-6):
    """d F_{k,axis} / d U_j of the oracle's lattice flux by central differences."""
    m = o.m_total
    J = np.zeros((m, m))
    for j in range(m):
        d = np.zeros(m); d[j] = h * max(1.0, abs(U[j]))
        Fp, _ = o.flux_source(U + d, A)
        Fm, _ = o.flux_source(U - d, A)
        J[:, j] = (Fp[:, axis] - Fm[:, axis]) / (2.0 * d[j])
    return J


def _grid_for(system, params, g_tau=4.0, lam=3.0, dx=0.01):
    return oracle.OracleGrid(system, 4, 4, 4 if system in ("nsf3d", "mhd3d", "hcnsf3d") else 1, dx, lam, params=params, g_tau=g_tau)


HYPERBOLIC = [   # (system, params with the dissipative coefficients at zero, state, conserved count)
    ("euler2d", [1.4], [1.3, 0.4, -0.9, 3.1], 4),
    ("swe2d", [9.81], [0.7, 0.3, -0.2], 3),
    ("swe2d_bathy", [9.81], [0.7, 0.3, -0.2], 3),
    ("inse2d", [1.7, 0.0], [1.1, 0.2, -0.3] + [0.0] * 4, 3),
    ("nsf2d", [1.4, 0.0, 0.0], [1.3, 0.4, -0.9, 3.1] + [0.0] * 8, 4),
    ("nsf3d", [1.4, 0.0, 0.0], [1.3, 0.4, -0.9, 0.5, 3.1] + [0.0] * 12, 5),
    ("hcnsf3d", [1.4, 0.0, 0.0, 1.0], [1.3, 0.4, -0.9, 0.5, 3.1] + [0.0] * 9, 5),
    ("mhd2d", [1.4, 0.0, 0.0, 0.0], [1.3, 0.4, -0.9, 3.5, 0.6, -0.3] + [0.0] * 12, 6),
]


@pytest.mark.parametrize("system,params,U,mc", HYPERBOLIC)
def test_p20_hyperbolic_speed_is_the_spectral_radius_of_the_flux_jacobian(system, params, U, mc):
    o = _grid_for(system, params)
    U = np.array(U, dtype=float)
    A = np.array([1.0, 0.0, 0.0, 0.0])[: max(o.n_aux, 1)]
    o.init_from_U(np.broadcast_to(U[:, None, None, None], o.shape_U).copy())
    s_axis, s_iso, s_diff = o.max_wave_speed()                      # lattice units: physical / lambda
    radii = []
    for axis in range(o.dim):
        J = _jacobian(o, U, A, axis)[:mc, :mc]                       # conserved block (trackers at zero, coefficients zero)
        radii.append(np.abs(np.linalg.eigvals(J)).max())
    assert s_axis == pytest.approx(max(radii), rel=1e-6)
    # isotropic bound: spectral radius of sum_a n_a A_a along the flow direction
    u = U[1:1 + o.dim] / U[0]
    nvec = u / np.linalg.norm(u)
    Jn = sum(nvec[a] * _jacobian(o, U, A, a)[:mc, :mc] for a in range(o.dim))
    r_n = np.abs(np.linalg.eigvals(Jn)).max()
    assert s_iso >= r_n * (1 - 1e-6)
    if system != "mhd2d":                                            # gas dynamics: |u| + c exactly; MHD: fast speed <= sqrt(a^2 + b^2)
        assert s_iso == pytest.approx(r_n, rel=1e-6)
    assert s_diff == 0.0
    o.close()


@pytest.mark.parametrize("system,params,U", [("allencahn2d", [0.01, 1.0], [0.3, 0.0, 0.0]), ("adr2d", [0.0, 0.0, 0.01, 1.0], [0.4, 0.0, 0.0])])
def test_p20_tracker_signal_speed_is_the_spectral_radius_for_pure_diffusion(system, params, U):
    """Parent/tracker pair [[0, -D_L], [-1/g_tau, 0]]: eigenvalues +- sqrt(D_L/g_tau) (from eq 2.3 L96 + eq 2.20)."""
    o = _grid_for(system, params, g_tau=6.0, lam=50.0)
    U = np.array(U, dtype=float)
    o.init_from_U(np.broadcast_to(U[:, None, None, None], o.shape_U).copy())
    s_axis, s_iso, s_diff = o.max_wave_speed()
    r = max(np.abs(np.linalg.eigvals(_jacobian(o, U, np.zeros(1), a))).max() for a in range(2))
    assert s_diff == pytest.approx(r, rel=1e-6) and s_axis == 0.0
    o.close()


@pytest.mark.parametrize("system,params,U", [
    ("nsf3d", [1.4, 2e-3, 1e-2], [1.3, 0.4, -0.9, 0.5, 3.1] + [0.01, -0.02, 0.0, 0.03, 0.0, 0.01, 0.0, 0.02, -0.01, 0.02, -0.01, 0.01]),
    ("nsf2d", [1.4, 2e-3, 1e-2], [1.3, 0.4, -0.9, 3.1] + [0.01, -0.02, 0.0, 0.03, 0.0, 0.01, 0.0, 0.02]),
    ("inse2d", [1.7, 5e-3], [1.1, 0.2, -0.3, 0.01, -0.02, 0.0, 0.03]),
    ("mhd3d", [1.4, 5e-3], [1.3, 0.4, -0.9, 0.5, 3.5, 0.6, -0.3, 0.2, 0.01, -0.02, 0.01]),
    ("mhd2d", [1.4, 2e-3, 1e-2, 5e-3], [1.3, 0.4, -0.9, 3.5, 0.6, -0.3] + [0.01, -0.02, 0.0, 0.03, 0.0, 0.01, 0.0, 0.02, -0.01, 0.02, -0.01, 0.01]),
])
def test_p20_check_speed_bounds_the_augmented_jacobian(system, params, U):
    """The speed the sub-characteristic check compares with c_s, max(out0, out1)/lambda + out2, is an upper bound of the
    spectral radius of the FULL augmented lattice Jacobian (hyperbolic part and tracker coupling together), and not a
    loose one (within a factor 2)."""
    o = _grid_for(system, params, g_tau=4.0, lam=4.0, dx=0.02)
    U = np.array(U, dtype=float)
    o.init_from_U(np.broadcast_to(U[:, None, None, None], o.shape_U).copy())
    s_axis, s_iso, s_diff = o.max_wave_speed()
    r = max(np.abs(np.linalg.eigvals(_jacobian(o, U, np.zeros(4), a))).max() for a in range(o.dim))
    bound = max(s_axis, s_iso) + s_diff
    assert s_diff > 0 and r <= bound * (1 + 1e-9) and bound <= 2.0 * r
    o.close()


def test_p20_elasticity_rest_state_speed():
    """The check uses the longitudinal speed of the linearisation about F = I (a constant although the material is nonlinear:
    stated limitation); at the rest state it is the spectral radius of the flux Jacobian."""
    o = _grid_for("elasticity2d", [1.0, 0.5, 1.0], lam=5.0)
    U = np.array([1.0, 0.0, 0.0, 1.0, 0.0, 0.0])
    o.init_from_U(np.broadcast_to(U[:, None, None, None], o.shape_U).copy())
    s_axis, _, _ = o.max_wave_speed()
    r = max(np.abs(np.linalg.eigvals(_jacobian(o, U, np.zeros(1), a))).max() for a in range(2))
    assert s_axis == pytest.approx(r, rel=1e-6) and s_axis == pytest.approx(math.sqrt(2.0) / 5.0, rel=1e-12)
    o.close()


# ------------------------------------------------------------------------------------------------ P11 on the configs
def _l2_errors(w, steps):
    g = oracle.OracleGrid.from_workload(w)
    g.init_from_U(w.initial_U())
    g.step(steps)
    U = g.read_U()
    _, t = g.time()
    Ue = g.exact_U(t)
    g.close()
    return [math.sqrt(((U[k] - Ue[k]) ** 2).sum() / (Ue[k] ** 2).sum()) for k in range(U.shape[0])]


def test_p11_c2_refinement_order():
    """configs[1] (flat-bottom SWE, manufactured forcing) at N = 64, 128, 256 to the time the config reaches at N = 512 after
    its 1000 steps: L2 order of h and hu in the paper's band."""
    ns, errs = (64, 128, 256), []
    for n in ns:
        errs.append(_l2_errors(W.c2_swe(n), 1000 * n // 512))
    for k in (0, 1):
        slope = -np.polyfit(np.log2(ns), np.log2([e[k] for e in errs]), 1)[0]
        assert 1.7 <= slope <= 2.5, (k, slope, errs)


def test_p11_c4_refinement_order_fp64():
    """The fp64 build of configs[3] (NSF 3D + 12 trackers, forcing on) at N = 16, 32, 64 to a fixed time: L2 order of the five
    conserved fields in the band."""
    ns, errs = (16, 32, 64), []
    for n in ns:
        errs.append(_l2_errors(W.c4_nsf3d(n, precision="f64"), 2 * n))
    for k in range(5):
        slope = -np.polyfit(np.log2(ns), np.log2([e[k] for e in errs]), 1)[0]
        assert 1.7 <= slope <= 2.5, (k, slope, [e[k] for e in errs])


# ------------------------------------------------------------------------------------------------ P21 config 3 against linear acoustics
def test_p21_c3_free_evolution_matches_linear_acoustics_at_small_amplitude():
    """configs[2] (Euler, u = 0, seeded smooth density / pressure perturbations) has no closed form at its amplitude 1e-2, but its
    linearisation has: with c^2 = gamma p0/rho0 = 1 every Fourier mode of the pressure is a standing wave dp_k(t) = dp_k(0) cos(c|k|t),
    the density follows as drho_k(t) = drho_k(0) + (cos(c|k|t) - 1) dp_k(0)/c^2 (the entropy part stays), the momentum is
    m_k(t) = -i k dp_k(0) sin(c|k|t)/(c|k|).  The oracle run of the SAME workload recipe at amplitude 1e-6 (nonlinear terms 1e-12)
    must follow it up to the scheme's own O(dx^2) + relaxation-diffusion error; run at two resolutions, the deviation falls."""
    devs = []
    for n in (64, 128):
        w = W.c3_euler(n, precision="f64")
        w.mms_params = [1e-6]                                   # amplitude of the seeded perturbations
        w.tau_R = 0.2
        U0 = w.initial_U()
        steps = int(round(0.3 / w.dt))
        U = oracle.run(w, steps=steps, U0=U0)
        t = steps * w.dt
        gamma = w.params[0]
        rho0, p0 = 1.0, 1.0 / gamma
        drho0 = U0[0, 0] - rho0
        dp0 = (gamma - 1.0) * U0[3, 0] - p0
        kx = 2 * np.pi * np.fft.fftfreq(n, d=w.dx)[None, :]
        ky = 2 * np.pi * np.fft.fftfreq(n, d=w.dx)[:, None]
        kk = np.sqrt(kx ** 2 + ky ** 2)
        ph = np.fft.fft2(dp0)
        cos_, sin_over = np.cos(kk * t), np.where(kk > 0, np.sin(kk * t) / np.where(kk > 0, kk, 1.0), t)
        dp_t = np.fft.ifft2(ph * cos_).real
        drho_t = drho0 + np.fft.ifft2(ph * (cos_ - 1.0)).real
        mx_t = np.fft.ifft2(-1j * kx * ph * sin_over).real
        u = U[1, 0] / U[0, 0]
        p = (gamma - 1.0) * (U[3, 0] - 0.5 * U[0, 0] * (u ** 2 + (U[2, 0] / U[0, 0]) ** 2))
        amp = np.abs(dp0).max()
        dev = max(np.abs(p - p0 - dp_t).max(), np.abs(U[0, 0] - rho0 - drho_t).max(), np.abs(U[1, 0] - mx_t).max()) / amp
        devs.append(dev)
    assert devs[1] < 0.02 and devs[1] < 0.45 * devs[0], devs      # second-order approach to the linear solution


# ------------------------------------------------------------------------------------------------ P22: dynamics of the round-2 systems
def _decay_rate(w, U0, steps, comp, shape_fn, x):
    g = oracle.OracleGrid.from_workload(w)
    if g.n_aux:
        g.set_aux(w.aux_fields(0.0))
    g.init_from_U(U0)
    s1 = steps // 4
    g.step(s1)
    a1 = 2.0 * np.abs((shape_fn(g.read_U()) * np.sin(K2PI * x)).mean())
    g.step(steps - s1)
    a2 = 2.0 * np.abs((shape_fn(g.read_U()) * np.sin(K2PI * x)).mean())
    g.close()
    return math.log(a1 / a2) / ((steps - s1) * w.dt)


def _chain_rule_system_state(system, n, dx, gamma, uy=None, rho=None, By=None):
    """nsf2d / mhd2d state on an (n, 2) grid varying in x: conserved fields + trackers = dx * analytic x-gradients of them."""
    x = np.arange(n) * dx
    one = np.ones((2, 1))
    rho = np.ones(n) if rho is None else rho
    uy = np.zeros(n) if uy is None else uy
    By = np.zeros(n) if By is None else By
    p0 = 1.0 / gamma
    E = p0 / (gamma - 1.0) + 0.5 * rho * uy ** 2 + 0.5 * By ** 2
    d = lambda a: np.real(np.fft.ifft(1j * 2 * np.pi * np.fft.fftfreq(n, d=dx) * np.fft.fft(a)))   # spectral d/dx (periodic, exact for these modes)
    cons = [rho, 0 * x, rho * uy, E] + ([0 * x, By] if system == "mhd2d" else [])
    M = (4 + 8) if system == "nsf2d" else (6 + 12)
    U = np.zeros((M, 1, 2, n))
    for k, c in enumerate(cons):
        U[k, 0] = c * one
        U[len(cons) + 2 * k, 0] = dx * d(c) * one              # G_{V,0} = dx d_x V ; G_{V,1} = 0
    return U, x


@pytest.mark.parametrize("system", ["nsf2d", "mhd2d"])
def test_p22_chain_rule_viscous_shear_decay(system):
    """u_y = A sin kx decays at nu k^2 (rate with mu minus rate without): the viscous stress reconstructed by the CHAIN RULE from
    the conserved-field trackers -- sign, mu_L scaling, the 1/rho factors."""
    n, A, gamma, mu = 128, 1e-3, 1.4, 5e-3
    mk = W.pin_nsf2d if system == "nsf2d" else W.pin_mhd2d
    rates = []
    for m_ in (0.0, mu):
        w = W.relabel(mk(n), ny=2, mms_id=0, params=[gamma, m_, 0.0] + ([0.0] if system == "mhd2d" else []),
                      lam=8.0, tau_R=20.0, g_tau=3.0, U_ref=[0.0] * (12 if system == "nsf2d" else 18))
        U0, x = _chain_rule_system_state(system, n, w.dx, gamma, uy=A * np.sin(K2PI * np.arange(n) * w.dx))
        rates.append(_decay_rate(w, U0, 1600, 2, lambda U: U[2, 0, 0] / U[0, 0, 0], x))
    assert rates[1] - rates[0] == pytest.approx(mu * K2PI ** 2, rel=0.05)


@pytest.mark.parametrize("system", ["nsf2d", "mhd2d"])
def test_p22_chain_rule_thermal_mode_decay(system):
    """Isobaric entropy mode decays at kappa k^2, kappa = K (gamma-1)/(gamma rho0): the heat flux -K grad T with grad T reconstructed by
    the chain rule from G_rho, G_m, G_E (and G_B)."""
    n, eps, gamma, K = 128, 1e-3, 1.4, 2e-2
    mk = W.pin_nsf2d if system == "nsf2d" else W.pin_mhd2d
    rates = []
    for K_ in (0.0, K):
        w = W.relabel(mk(n), ny=2, mms_id=0, params=[gamma, 0.0, K_] + ([0.0] if system == "mhd2d" else []),
                      lam=8.0, tau_R=20.0, g_tau=3.0, U_ref=[0.0] * (12 if system == "nsf2d" else 18))
        xs = np.arange(n) * w.dx
        U0, x = _chain_rule_system_state(system, n, w.dx, gamma, rho=1.0 - eps * np.sin(K2PI * xs))

        def entropy(U):
            rho = U[0, 0, 0]
            p = (gamma - 1.0) * (U[3, 0, 0] - 0.5 * (U[1, 0, 0] ** 2 + U[2, 0, 0] ** 2) / rho)
            return np.log(gamma * p) - gamma * np.log(rho)
        rates.append(_decay_rate(w, U0, 1600, 0, entropy, x))
    assert rates[1] - rates[0] == pytest.approx(K * (gamma - 1.0) / gamma * K2PI ** 2, rel=0.05)


def test_p22_mhd2d_resistive_decay():
    """B_y = A sin kx decays at eta k^2: the resistive flux -eta G_B of the induction equation of the 2D system (eq 3.25)."""
    n, A, gamma, eta = 128, 1e-3, 1.4, 5e-3
    rates = []
    for e_ in (0.0, eta):
        w = W.relabel(W.pin_mhd2d(n), ny=2, mms_id=0, params=[gamma, 0.0, 0.0, e_], lam=8.0, tau_R=20.0, g_tau=3.0, U_ref=[0.0] * 18)
        U0, x = _chain_rule_system_state("mhd2d", n, w.dx, gamma, By=A * np.sin(K2PI * np.arange(n) * w.dx))
        rates.append(_decay_rate(w, U0, 1600, 5, lambda U: U[5, 0, 0], x))
    assert rates[1] - rates[0] == pytest.approx(eta * K2PI ** 2, rel=0.05)


def test_p22_hcnsf_drag_relaxes_towards_the_solid_velocity_exactly():
    """Uniform state, uniform prescribed fields: the only active term is the drag (1-alpha)/eta (rho u_s - rho u) (eq 3.27).
    The scheme adds dt S to the zeroth moment each step, so m_n = rho u_s + (m_0 - rho u_s)(1 - dt (1-alpha)/eta)^n EXACTLY; the
    energy follows dE = sum of dt S_m . u.  alpha = 1 switches the drag off."""
    w = W.hcnsf3d(4, precision="f64")
    gamma, mu, kap, eta = w.params
    for alpha in (1.0, 0.35):
        us = np.array([0.2, -0.1, 0.05])
        A = np.zeros((4, 4, 4, 4)); A[0] = alpha
        for a in range(3):
            A[1 + a] = us[a]
        U0 = np.zeros((14, 4, 4, 4))
        rho, u0 = 1.1, np.array([0.3, 0.1, -0.2])
        U0[0] = rho
        for a in range(3):
            U0[1 + a] = rho * u0[a]
        U0[4] = 1.0 / (gamma - 1.0) + 0.5 * rho * (u0 ** 2).sum()
        g = oracle.OracleGrid.from_workload(w)
        g.set_aux(A); g.init_from_U(U0); g.step(25)
        U = g.read_U(); g.close()
        q = 1.0 - w.dt * (1.0 - alpha) / eta
        want_m = rho * us + (rho * u0 - rho * us) * q ** 25
        assert np.allclose(U[1:4, 0, 0, 0], want_m, rtol=1e-12, atol=1e-15)
        assert np.allclose(U[0], rho, rtol=1e-14) and np.abs(U[5:]).max() < 1e-15        # no density change, trackers stay zero
        E, m = U0[4, 0, 0, 0], rho * u0.copy()
        for _ in range(25):                                                               # dE = dt S_m . u, step by step
            S = w.dt * (1.0 - alpha) / eta * (rho * us - m)
            E += (S * m / rho).sum(); m = m + S
        assert U[4, 0, 0, 0] == pytest.approx(E, rel=1e-13)


def test_p22_hcnsf_porosity_scales_the_viscous_decay():
    """u_y = A sin kx with uniform alpha and no drag (u_s = u would need eta -> inf: the drag is removed by alpha-independent choice
    eta = 1e30): decay rate(alpha, mu) - rate(alpha, 0) = alpha nu k^2 -- the factor alpha on tau, and the halves of the symmetric
    tracker sym(I (x) u)/tau_grad (a missing 1/2 would give half / twice the rate)."""
    n, A, gamma, mu = 128, 1e-3, 1.4, 5e-3
    for alpha in (1.0, 0.5):
        rates = []
        for m_ in (0.0, mu):
            w = W.relabel(W.hcnsf3d(n, ny=2, nz=2, precision="f64"), params=[gamma, m_, 0.0, 1e30], lam=8.0, tau_R=20.0, g_tau=3.0, U_ref=[0.0] * 14)
            x = np.arange(n) * w.dx
            one = np.ones((2, 2, 1))
            U0 = np.zeros((14, 2, 2, n))
            uy = A * np.sin(K2PI * x)
            U0[0] = 1.0; U0[2] = uy * one
            U0[4] = ((1.0 / gamma) / (gamma - 1.0) + 0.5 * uy ** 2) * one
            U0[8] = w.dx * 0.5 * A * K2PI * np.cos(K2PI * x) * one            # D_xy = (d_x u_y + d_y u_x)/2
            Aux = np.zeros((4, 2, 2, n)); Aux[0] = alpha
            g = oracle.OracleGrid.from_workload(w)
            g.set_aux(Aux); g.init_from_U(U0)
            g.step(400); a1 = 2.0 * np.abs((g.read_U()[2, 0, 0] * np.sin(K2PI * x)).mean())
            g.step(1200); a2 = 2.0 * np.abs((g.read_U()[2, 0, 0] * np.sin(K2PI * x)).mean())
            g.close()
            rates.append(math.log(a1 / a2) / (1200 * w.dt))
        assert rates[1] - rates[0] == pytest.approx(alpha * mu * K2PI ** 2, rel=0.05)
