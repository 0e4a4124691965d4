// oracle/mms_fields.hpp -- TEST INFRASTRUCTURE (CPU oracle). Not part of the product path.
//
// Exact manufactured fields Q_exact(x, t) of the systems that carry MMS forcing, as jets, and the
// manufactured source of eq (4.1), formed for the AUGMENTED system (trackers
// forced too, with G_exact = grad V_exact; SURVEY.md §8(c) reading A5, confirmed on the ADR row of
// Table 2).
//   burgers2d mms 1 : eq (SM5.1), A = mms_par[0] (Table SM3: 1.3)
//   euler2d   mms 1 : eq (SM5.2), non-dimensional rho0 = c_s = 1 (reading A9)
//   adr2d     mms 1 : eq (SM5.7), Table SM8
//   swe2d     mms 1 : BASELINE.json configs[1] fields, mms_par = {A_h, A_u, h0}
//   nsf3d     mms 1 : BASELINE.json configs[3] fields, mms_par = {U0, A_rho, rho0, p0}
//   urf2d     mms 1 : eq (SM5.4)
//   allencahn2d mms 1 : eq (SM5.8); Table SM9 L1316 (gamma = 0.01, r = 1)
//   inse2d    mms 1 : eq (SM5.9), PAPER.md:L1330-L1334 (Taylor-Green vortex), mms_par = {U, rho0}
//   elasticity2d mms 1 : eq (SM5.6)
//   nsf2d     mms 1 : eq (SM5.10)
//   swe2d_bathy mms 1 : eq (SM5.3), PAPER.md:L1200-L1207 with the static bed z_b of L1198
//   mhd2d     mms 1 : SM5.12 text
//   maxwell2d mms 1 : eq (SM5.5), PAPER.md:L1248-L1254 (k_x = 2 pi, k_y = 4 pi, A = 1/2, omega = 4)
#pragma once
#include "jets.hpp"
#include "systems.hpp"

namespace orc {

constexpr double PI = 3.14159265358979323846;

// Q[k] (value + first derivatives in t,x,y,z) of the exact augmented state at one point.
// returns false if (sys, mms_id) has no manufactured solution.
inline bool exact_state(int sys, int mms_id, const Scaling& sc, const double* mp,
                        double t_, double x_, double y_, double z_, J1* Q) {
    if (mms_id != 1) return false;
    const J2 t = J2::variable(0, t_), x = J2::variable(1, x_), y = J2::variable(2, y_), z = J2::variable(3, z_);
    const double k = 2.0 * PI;
    switch (sys) {
    case SYS_BURGERS2D: {
        J2 u = mp[0] * sin(k * x) * sin(k * y) * cos(t);
        Q[0] = lower(u);
        return true;
    }
    case SYS_EULER2D: {
        const double gamma = sc.par[0], rho0 = 1.0, cs = 1.0, p0 = rho0 * cs * cs / gamma, u0 = 3.0 * cs, v0 = 3.0 * cs;
        J2 drho = 0.3 * rho0 * sin(k * x) * cos(k * y) * cos(t);
        J2 du = 0.3 * cs * cos(k * x) * sin(k * y) * sin(t);
        J2 dv = 0.3 * cs * sin(k * x) * sin(k * y) * sin(t);
        J2 dp = cs * cs * drho + 0.2 * p0 * cos(k * x) * sin(k * y) * sin(t);
        J2 rho = rho0 + drho, u = u0 + du, v = v0 + dv, p = p0 + dp;
        J2 E = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v);
        Q[0] = lower(rho); Q[1] = lower(rho * u); Q[2] = lower(rho * v); Q[3] = lower(E);
        return true;
    }
    case SYS_SWE2D: {
        const double Ah = mp[0], Au = mp[1], h0 = mp[2];
        J2 h = h0 + Ah * sin(k * x) * cos(k * y) * cos(t);
        J2 u = Au * cos(k * x) * sin(k * y) * cos(t);
        J2 v = Au * sin(k * x) * sin(k * y) * sin(t);
        Q[0] = lower(h); Q[1] = lower(h * u); Q[2] = lower(h * v);
        return true;
    }
    case SYS_ADR2D: {
        const double u0 = sc.par[0], u1 = sc.par[1];
        J2 c = 0.5 * sin(k * (x - u0 * t)) * cos(k * (y - u1 * t)) * exp(-t) + 0.5;
        Q[0] = lower(c);
        Q[1] = sc.dx * diff(c, 1);
        Q[2] = sc.dx * diff(c, 2);
        return true;
    }
    case SYS_NSF3D: {
        const double gamma = sc.par[0], mu = sc.par[1];
        const double U0 = mp[0], Ar = mp[1], rho0 = mp[2], p0 = mp[3];
        J2 D = exp((-3.0 * (mu / rho0) * k * k) * t);
        J2 sx = sin(k * x), cx = cos(k * x), sy = sin(k * y), cy = cos(k * y), sz = sin(k * z), cz = cos(k * z);
        J2 u[3] = {U0 * sx * cy * cz * D, -U0 * cx * sy * cz * D, 0.5 * U0 * cx * cy * sz * D};
        J2 p = p0 + (rho0 * U0 * U0 / 16.0) * (cos(2.0 * k * x) + cos(2.0 * k * y)) * (cos(2.0 * k * z) + 2.0) * D * D;
        J2 rho = rho0 * (1.0 + Ar * sx * sy * cz * cos(t));
        J2 Tm = p / rho;
        J2 E = p / (gamma - 1.0) + 0.5 * rho * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        Q[0] = lower(rho);
        for (int a = 0; a < 3; ++a) Q[1 + a] = lower(rho * u[a]);
        Q[4] = lower(E);
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) Q[5 + 3 * a + b] = sc.dx * diff(u[a], 1 + b);
        for (int b = 0; b < 3; ++b) Q[14 + b] = sc.dx * diff(Tm, 1 + b);
        return true;
    }
    case SYS_URF2D: {
        Q[0] = lower(0.4 * sin(k * x) * sin(k * y) * cos(t) + 3.0);
        Q[1] = lower(0.4 * cos(k * x) * cos(k * y) * sin(t) + 1.2);
        Q[2] = lower(0.4 * sin(k * x) * sin(k * y) * sin(t) + 1.2);
        return true;
    }
    case SYS_ALLENCAHN2D: {
        J2 phi = 0.7 * sin(k * x) * cos(k * y) * cos(t);          // eq (SM5.8)
        Q[0] = lower(phi);
        Q[1] = sc.dx * diff(phi, 1);
        Q[2] = sc.dx * diff(phi, 2);
        return true;
    }
    case SYS_INSE2D: {
        // eq (SM5.9): 2D Taylor-Green vortex; mp = {U, rho0}; nu = mu/rho0
        const double cs = sc.par[0], U0 = mp[0], rho0 = mp[1], nu = sc.par[1] / rho0;
        J2 D = exp((-2.0 * (nu / cs) * k * k) * t);
        J2 u = -U0 * cos(k * x) * sin(k * y) * D;
        J2 v = U0 * sin(k * x) * cos(k * y) * D;
        J2 p = (-0.25 * rho0 * U0 * U0) * (cos(2.0 * k * x) + cos(2.0 * k * y)) * D * D;
        J2 rho = rho0 + p / (cs * cs);
        J2 mx = rho * u, my = rho * v;
        Q[0] = lower(rho); Q[1] = lower(mx); Q[2] = lower(my);
        Q[3] = sc.dx * diff(mx, 1); Q[4] = sc.dx * diff(mx, 2);
        Q[5] = sc.dx * diff(my, 1); Q[6] = sc.dx * diff(my, 2);
        return true;
    }
    case SYS_ELASTICITY2D: {
        // eq (SM5.6): displacement potential w, F = I + grad w, v = d_t w; A = 0.06
        const double A = 0.06, rho0 = sc.par[0];
        J2 w0 = A * (sin(k * x) * sin(k * y) * cos(t) + 0.5 * sin(k * x) * cos(k * y) * sin(t) + 0.25 * cos(k * (x + y)) * cos(t));
        J2 w1 = A * (cos(k * x) * cos(k * y) * sin(t) + 0.5 * cos(k * x) * sin(k * y) * cos(t) + 0.25 * sin(k * (x - y)) * sin(t));
        Q[0] = 1.0 + diff(w0, 1); Q[1] = diff(w0, 2);
        Q[2] = diff(w1, 1);       Q[3] = 1.0 + diff(w1, 2);
        Q[4] = rho0 * diff(w0, 0); Q[5] = rho0 * diff(w1, 0);
        return true;
    }
    case SYS_NSF2D: {
        // eq (SM5.10), non-dimensional rho0 = c_s = 1 (reading A9): u0 = 3, v0 = 2, p0 = 1/gamma
        const double gamma = sc.par[0], p0 = 1.0 / gamma;
        J2 drho = 0.2 * sin(k * x) * cos(k * y) * cos(t);
        J2 rho = 1.0 + drho;
        J2 u = 3.0 + 0.2 * cos(k * x) * sin(k * y) * sin(t);
        J2 v = 2.0 + 0.15 * sin(k * x) * sin(k * y) * cos(t);
        J2 p = p0 + drho + (0.2 * p0) * cos(k * x) * sin(k * y) * sin(t);
        J2 V[4] = {rho, rho * u, rho * v, p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v)};
        for (int q = 0; q < 4; ++q) {
            Q[q] = lower(V[q]);
            Q[4 + 2 * q + 0] = sc.dx * diff(V[q], 1);
            Q[4 + 2 * q + 1] = sc.dx * diff(V[q], 2);
        }
        return true;
    }
    case SYS_SWE2D_BATHY: {
        // eq (SM5.3): h = h0 + A_h sin sin cos t, hu0 = m0 + A_m cos cos sin t, hu1 = m0 + A_m sin sin sin t;
        // mp = {h0, A_h, m0, A_m, A_zb, w} (paper: 0.1, 0.04, 0.03, 0.02, 0.01 before non-dimensionalisation; w = frequency of
        // the time factors in the non-dimensional time, A25)
        const double h0 = mp[0], Ah = mp[1], m0 = mp[2], Am = mp[3], w = mp[5];
        Q[0] = lower(h0 + Ah * sin(k * x) * sin(k * y) * cos(w * t));
        Q[1] = lower(m0 + Am * cos(k * x) * cos(k * y) * sin(w * t));
        Q[2] = lower(m0 + Am * sin(k * x) * sin(k * y) * sin(w * t));
        return true;
    }
    case SYS_MHD2D: {
        // eq (SM5.12 text), non-dimensional rho0 = c_s = 1 (reading A9): u0 = v0 = 3, B0 = 0.5, p0 = 1/gamma
        const double gamma = sc.par[0], p0 = 1.0 / gamma;
        J2 drho = 0.3 * sin(k * x) * cos(k * y) * cos(t);
        J2 rho = 1.0 + drho;
        J2 p = p0 + drho + (0.2 * p0) * cos(k * x) * sin(k * y) * sin(t);
        J2 u = 3.0 + 0.3 * cos(k * x) * sin(k * y) * sin(t);
        J2 v = 3.0 + 0.3 * sin(k * x) * sin(k * y) * sin(t);
        J2 Bx = 0.5 - 0.3 * cos(k * x) * sin(k * y) * sin(t);
        J2 By = 0.5 + 0.3 * sin(k * x) * cos(k * y) * sin(t);
        J2 V[6] = {rho, rho * u, rho * v, p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v) + 0.5 * (Bx * Bx + By * By), Bx, By};
        for (int q = 0; q < 6; ++q) {
            Q[q] = lower(V[q]);
            Q[6 + 2 * q + 0] = sc.dx * diff(V[q], 1);
            Q[6 + 2 * q + 1] = sc.dx * diff(V[q], 2);
        }
        return true;
    }
    case SYS_MAXWELL2D: {
        const double A = 0.5, kx = 2.0 * PI, ky = 4.0 * PI, om = 4.0;
        Q[0] = lower(A * sin(kx * x) * sin(ky * y) * cos(om * t));
        Q[1] = lower(A * sin(kx * x) * cos(ky * y) * sin(om * t));
        Q[2] = lower((-A * kx / ky) * cos(kx * x) * sin(ky * y) * sin(om * t));
        return true;
    }
    }
    return false;
}

// Prescribed coefficient fields of the manufactured cases, as jets (their gradients enter where the flux holds them).
inline void exact_aux(int sys, const Scaling& sc, const double* mp, double t_, double x_, double y_, double z_, J1* A) {
    (void)sc; (void)t_; (void)z_;
    const J2 x = J2::variable(1, x_), y = J2::variable(2, y_);
    const double k = 2.0 * PI;
    if (sys == SYS_SWE2D_BATHY) {
        // static bathymetry z_b = A_zb sin(2 pi x0) cos(2 pi x1); the field handed to the scheme is its slope
        J2 zb = mp[4] * sin(k * x) * cos(k * y);
        A[0] = diff(zb, 1);
        A[1] = diff(zb, 2);
    }
}

// Lattice manufactured source at one point:
//   s_mms[k] = dt * d_t Q_k + dx * sum_a d_a F_k,a(Q_exact) - S_k(Q_exact)      (eq 4.1 in lattice units;
//   F = (dt/dx) Phi and S = dt * S_phys, so this is dt * [d_t Q + div Phi - S_phys].)
inline bool mms_source(int sys, int mms_id, const Scaling& sc, const double* mp,
                       double t, double x, double y, double z, double* s_mms) {
    J1 Q[MAXM], F[MAXM * 3], S[MAXM], A[8];
    if (!exact_state(sys, mms_id, sc, mp, t, x, y, z, Q)) return false;
    exact_aux(sys, sc, mp, t, x, y, z, A);
    flux_source<J1>(sys, Q, A, sc, F, S);
    const int m = sys_info(sys).m_total;
    for (int k = 0; k < m; ++k)
        s_mms[k] = sc.dt * Q[k].d[0] + sc.dx * (F[k * 3 + 0].d[1] + F[k * 3 + 1].d[2] + F[k * 3 + 2].d[3]) - S[k].v;
    return true;
}

}  // namespace orc
