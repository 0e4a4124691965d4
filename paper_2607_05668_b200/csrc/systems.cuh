// systems.cuh -- per-system lattice flux F_k = (dt/dx) Phi_k(Q+) and source s_k = dt S_k(Q+), in delta form.
//
// Every system is written ONCE for the state split Q = Q0 + dQ of eq (2.23): the
// kernels hand in dQ (the zeroth moments of the shifted populations f*) and get back
//     dF_k = F_k(Q0 + dQ) - F_k(Q0)          and        s_k(Q0 + dQ)
// with every dF term O(dQ): products of two O(1) backgrounds are cancelled on paper, not in fp32
// (SURVEY.md Appendix B).  With Q0 = 0 (plain fp64 form) the same code is the plain flux.
// Host-derived reference constants arrive in KParams::cst (filled by derive_constants in lbmk_api.cu):
//   hydrodynamic systems  cst[0..2] = u0 = m0/rho0,  cst[3] = p0,  cst[4] = E0 + p0,  cst[5] = T0 = p0/rho0
//   SWE                   cst[0..1] = u0 = m0/h0
//   ultrarelativistic     cst[0..1] = v0,  cst[2] = sqrt(D0),  cst[3] = p0,  cst[4] = W0 = 2 E0 + sqrt(D0)
// Trackers are in lattice units G^L = dx grad V: F_G[b][j] = G_b u_j/lambda - delta_jb V/g_tau,
// s_G = -G/g_tau (eq 2.3; tau_grad = g_tau dt, L106); a physical diffusivity D enters the
// parent's flux as D_L = D dt/dx^2.
//
// Interface of a system S<R>:
//   ID, D (dimension), M (components), MC (conserved), Ctx (primitives shared by all components)
//   setup(Ctx&, dQ[M], P)                 once per node
//   flux<k>(Ctx, dQ, P, F[D], S)          lattice flux columns and source of component k
//   wave(Q[M] full state, P, out[3])      physical |u_a|+c_a max, |u|+c, lattice diffusive signal speed
// Systems with prescribed per-node coefficient fields (the bed slope of eq 3.5) also declare
//   NA (their number), set_aux(Ctx&, A[NA]) -- called before setup with this node's values -- and default_aux(Ctx&).
#pragma once
#include "cascade_generated.cuh"
#include "common.cuh"

namespace lbmk {

enum { SYS_ADVECTION2D = 0, SYS_BURGERS2D = 1, SYS_SWE2D = 2, SYS_EULER2D = 3, SYS_ADR2D = 4, SYS_NSF3D = 5, SYS_MHD3D = 6,
       SYS_URF2D = 7, SYS_MAXWELL2D = 8, SYS_ALLENCAHN2D = 9, SYS_INSE2D = 10, SYS_ELASTICITY2D = 11, SYS_NSF2D = 12,
       SYS_SWE2D_BATHY = 13, SYS_HCNSF3D = 14, SYS_MHD2D = 15 };

// ------------------------------------------------------------------------------------------ advection
// Phi = (a_x U, a_y U); par = {a_x, a_y}
template <class R> struct SysAdvection2D {
    static constexpr int ID = SYS_ADVECTION2D, D = 2, M = 1, MC = 1;
    static constexpr bool LINEAR = true;     // flux = one product per entry: no FMA-contraction freedom, every kernel gives the same bits
    using Mms = void;
    struct Ctx {};
    __device__ __forceinline__ static void setup(Ctx&, const R (&)[M], const KParams<R>&) {}
    template <int k> __device__ __forceinline__ static void flux(const Ctx&, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        F[0] = (P.par[0] * P.il) * dQ[0];
        F[1] = (P.par[1] * P.il) * dQ[0];
        S = R(0);
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double ax = fabs(P.par[0]), ay = fabs(P.par[1]);
        out[0] = fmax(ax, ay); out[1] = sqrt(ax * ax + ay * ay); out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ Burgers
// eq (3.1)-(3.2): Phi = (u^2/2, u^2/2);  delta form du (u0 + du/2)
template <class R> struct SysBurgers2D {
    static constexpr int ID = SYS_BURGERS2D, D = 2, M = 1, MC = 1;
    using Mms = Mms_burgers2d;
    struct Ctx {};
    __device__ __forceinline__ static void setup(Ctx&, const R (&)[M], const KParams<R>&) {}
    template <int k> __device__ __forceinline__ static void flux(const Ctx&, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        const R h = P.il * (dQ[0] * (P.ref[0] + R(0.5) * dQ[0]));
        F[0] = h; F[1] = h;
        S = R(0);
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double a = fabs(Q[0]);      // f'(u) = u on both axes
        out[0] = a; out[1] = sqrt(2.0) * a; out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ shallow water
// eq (3.6), flat bottom; par = {g}; Q = (h, hu, hv)
template <class R> struct SysSwe2D {
    static constexpr int ID = SYS_SWE2D, D = 2, M = 3, MC = 3;
    using Mms = Mms_swe2d;
    struct Ctx { R u[2], du[2], dP; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R h = P.ref[0] + dQ[0];
        const R rh = R(1) / h;
        for (int a = 0; a < 2; ++a) {
            c.du[a] = (dQ[1 + a] - P.cst[a] * dQ[0]) * rh;     // u - u0 = (dm - u0 dh)/h
            c.u[a] = P.cst[a] + c.du[a];
        }
        c.dP = R(0.5) * P.par[0] * dQ[0] * (R(2) * P.ref[0] + dQ[0]);   // g/2 (h^2 - h0^2)
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        S = R(0);
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2];
        } else {
            constexpr int a = k - 1;
            for (int j = 0; j < 2; ++j) {
                R v = dQ[1 + a] * c.u[j] + P.ref[1 + a] * c.du[j];      // m_a u_j - m0_a u0_j
                if (j == a) v += c.dP;
                F[j] = P.il * v;
            }
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double cc = sqrt(P.par[0] * Q[0]), u = Q[1] / Q[0], v = Q[2] / Q[0];
        out[0] = fmax(fabs(u), fabs(v)) + cc; out[1] = sqrt(u * u + v * v) + cc; out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ Euler 2D
// eq (3.4); p = (gamma-1)(E - rho|u|^2/2); par = {gamma}; Q = (rho, mx, my, E)
template <class R> struct SysEuler2D {
    static constexpr int ID = SYS_EULER2D, D = 2, M = 4, MC = 4;
    using Mms = Mms_euler2d;
    struct Ctx { R u[2], du[2], dp; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R rho = P.ref[0] + dQ[0];
        const R r = R(1) / rho;
        R dke = R(0);
        for (int a = 0; a < 2; ++a) {
            c.du[a] = (dQ[1 + a] - P.cst[a] * dQ[0]) * r;
            c.u[a] = P.cst[a] + c.du[a];
            dke += dQ[1 + a] * c.u[a] + P.ref[1 + a] * c.du[a];         // m.u - m0.u0
        }
        c.dp = (P.par[0] - R(1)) * (dQ[3] - R(0.5) * dke);
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        S = R(0);
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2];
        } else if constexpr (k == 3) {
            for (int j = 0; j < 2; ++j) F[j] = P.il * ((dQ[3] + c.dp) * c.u[j] + P.cst[4] * c.du[j]);
        } else {
            constexpr int a = k - 1;
            for (int j = 0; j < 2; ++j) {
                R v = dQ[1 + a] * c.u[j] + P.ref[1 + a] * c.du[j];
                if (j == a) v += c.dp;
                F[j] = P.il * v;
            }
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double u = Q[1] / Q[0], v = Q[2] / Q[0];
        const double p = (P.par[0] - 1.0) * (Q[3] - 0.5 * Q[0] * (u * u + v * v));
        const double cc = sqrt(P.par[0] * p / Q[0]);
        out[0] = fmax(fabs(u), fabs(v)) + cc; out[1] = sqrt(u * u + v * v) + cc; out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ scalar ADR
// eq (3.17); SM4.7 L908-L926; par = {u_x, u_y, D, R}; Q = (c, G^L_x, G^L_y)
template <class R> struct SysAdr2D {
    static constexpr int ID = SYS_ADR2D, D = 2, M = 3, MC = 1;
    using Mms = Mms_adr2d;
    struct Ctx {};
    __device__ __forceinline__ static void setup(Ctx&, const R (&)[M], const KParams<R>&) {}
    template <int k> __device__ __forceinline__ static void flux(const Ctx&, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        const R ax = P.par[0] * P.il, ay = P.par[1] * P.il;
        if constexpr (k == 0) {
            const R DL = P.par[2] * P.dL;
            F[0] = ax * dQ[0] - DL * dQ[1];
            F[1] = ay * dQ[0] - DL * dQ[2];
            const R c = P.ref[0] + dQ[0];
            S = P.dt * P.par[3] * c * (R(1) - c);                       // reaction at the full state
        } else {
            constexpr int b = k - 1;
            F[0] = ax * dQ[k]; F[1] = ay * dQ[k];
            F[b] -= dQ[0] * P.inv_gtau;
            S = -(P.ref[k] + dQ[k]) * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double ax = fabs(P.par[0]), ay = fabs(P.par[1]);
        out[0] = fmax(ax, ay); out[1] = sqrt(ax * ax + ay * ay);
        out[2] = sqrt(P.par[2] * P.dL * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ Allen-Cahn
// eq (3.18)-(3.19); SM4.8 L928-L945; par = {gamma, r}; Q = (phi, G^L_x, G^L_y)
template <class R> struct SysAllenCahn2D {
    static constexpr int ID = SYS_ALLENCAHN2D, D = 2, M = 3, MC = 1;
    using Mms = Mms_allencahn2d;
    struct Ctx {};
    __device__ __forceinline__ static void setup(Ctx&, const R (&)[M], const KParams<R>&) {}
    template <int k> __device__ __forceinline__ static void flux(const Ctx&, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            const R gL = P.par[0] * P.dL;
            F[0] = -gL * dQ[1];
            F[1] = -gL * dQ[2];
            const R phi = P.ref[0] + dQ[0];
            S = (P.dt * P.par[1]) * (phi - phi * phi * phi);            // bistable reaction at the full state
        } else {
            constexpr int b = k - 1;
            F[0] = R(0); F[1] = R(0);
            F[b] = -dQ[0] * P.inv_gtau;
            S = -(P.ref[k] + dQ[k]) * P.inv_gtau;
        }
    }
    __device__ static void wave(const double*, const KParams<double>& P, double* out) {
        out[0] = 0.0; out[1] = 0.0; out[2] = sqrt(P.par[0] * P.dL * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ weakly compressible NSE
// eq (3.21)-(3.22); SM4.9 L947-L959; par = {c_s_phys, mu};
// Q = (rho, m_x, m_y, G^L_ab = dx d_b m_a [index 3+2a+b]).  Reference: rho0 free, m0 = 0, trackers 0 (host-checked).
//   dF_rho,j = m_j/lam;  dF_ma,j = (m_a u_j + delta_aj c_s^2 drho)/lam - (mu_L/rho)(G_aj + G_ja)
//   dF_Gab,j = G_ab u_j/lam - delta_jb m_a/g_tau;  s_G = -G/g_tau
template <class R> struct SysInse2D {
    static constexpr int ID = SYS_INSE2D, D = 2, M = 7, MC = 3;
    using Mms = Mms_inse2d;
    struct Ctx { R ul[2], nuL; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R r = R(1) / (P.ref[0] + dQ[0]);
        c.ul[0] = dQ[1] * r * P.il; c.ul[1] = dQ[2] * r * P.il;
        c.nuL = P.par[1] * P.dL * r;
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2]; S = R(0);
        } else if constexpr (k <= 2) {
            constexpr int a = k - 1;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                R v = dQ[1 + a] * c.ul[j] - c.nuL * (dQ[3 + 2 * a + j] + dQ[3 + 2 * j + a]);
                if (a == j) v += (P.il * P.par[0] * P.par[0]) * dQ[0];
                F[j] = v;
            }
            S = R(0);
        } else {
            constexpr int a = (k - 3) / 2, b = (k - 3) % 2;
            F[0] = dQ[k] * c.ul[0]; F[1] = dQ[k] * c.ul[1];
            F[b] -= dQ[1 + a] * P.inv_gtau;
            S = -dQ[k] * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double u = Q[1] / Q[0], v = Q[2] / Q[0], cc = P.par[0];
        out[0] = fmax(fabs(u), fabs(v)) + cc; out[1] = sqrt(u * u + v * v) + cc;
        out[2] = sqrt(2.0 * P.par[1] * P.dL / Q[0] * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ finite-strain elasticity
// eq (3.13)-(3.15); SM4.6 L865-L897: Q = (F_00, F_01, F_10, F_11, rho0 v_0, rho0 v_1);
// d_t F_ij - d_j v_i = 0, d_t (rho0 v_i) - d_k P_ik = 0, P = mu_s (F - F^-T) + lambda_s ln(J) F^-T; par = {rho0, mu_s, lambda_s}.
// Reference: the rest configuration F = I, v = 0 (P(I) = 0) or none.  With d = F - I:
//   dJ = d00 + d11 + d00 d11 - d01 d10,  F^-T = [[1+d11, -d10], [-d01, 1+d00]]/J,  I - F^-T = [[dJ-d11, d10], [d01, dJ-d00]]/J,
//   P = mu_s (d + (I - F^-T)) + lambda_s log1p(dJ) F^-T   -- every term O(d).
template <class R> struct SysElasticity2D {
    static constexpr int ID = SYS_ELASTICITY2D, D = 2, M = 6, MC = 6;
    using Mms = Mms_elasticity2d;
    struct Ctx { R P[2][2], vl[2]; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R d00 = (P.ref[0] - R(1)) + dQ[0], d01 = P.ref[1] + dQ[1], d10 = P.ref[2] + dQ[2], d11 = (P.ref[3] - R(1)) + dQ[3];
        const R dJ = d00 + d11 + d00 * d11 - d01 * d10;
        const R iJ = R(1) / (R(1) + dJ);
        const R lJ = P.par[2] * log1p(dJ), mu = P.par[1];
        const R T00 = (R(1) + d11) * iJ, T01 = -d10 * iJ, T10 = -d01 * iJ, T11 = (R(1) + d00) * iJ;    // F^-T
        c.P[0][0] = mu * (d00 + (dJ - d11) * iJ) + lJ * T00;
        c.P[0][1] = mu * (d01 + d10 * iJ) + lJ * T01;
        c.P[1][0] = mu * (d10 + d01 * iJ) + lJ * T10;
        c.P[1][1] = mu * (d11 + (dJ - d00) * iJ) + lJ * T11;
        const R ir = P.il / P.par[0];
        c.vl[0] = (P.ref[4] + dQ[4]) * ir; c.vl[1] = (P.ref[5] + dQ[5]) * ir;
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&)[M], const KParams<R>& P, R (&F)[D], R& S) {
        S = R(0);
        if constexpr (k < 4) {
            constexpr int i = k / 2, j = k % 2;
            F[0] = R(0); F[1] = R(0);
            F[j] = -c.vl[i];
        } else {
            constexpr int i = k - 4;
            F[0] = -P.il * c.P[i][0]; F[1] = -P.il * c.P[i][1];
        }
    }
    __device__ static void wave(const double*, const KParams<double>& P, double* out) {
        const double cp = sqrt((P.par[2] + 2.0 * P.par[1]) / P.par[0]);      // rest-state longitudinal speed
        out[0] = cp; out[1] = cp; out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ compressible NSF 2D
// eq (3.23)-(3.24); Listing 2; cascade on the CONSERVED fields (N = 4 + 8, SM4.10 L961):
// Q = (rho, m0, m1, E, G^L_{V,b} = dx d_b V [index 4 + 2 v + b], V = rho, m0, m1, E); par = {gamma, mu, K}.
// Derived gradients by the chain rule: d_b u_a = (G_{ma,b} - u_a G_{rho,b})/rho,
//   d_b p = (gamma-1)(G_{E,b} - u.G_{m,b} + |u|^2/2 G_{rho,b}),  d_b T = (d_b p - T G_{rho,b})/rho,  T = p/rho.
// Reference: (rho0, m0, E0) free (moving reference as in Euler 2D), trackers 0 (host-checked).
template <class R> struct SysNsf2D {
    static constexpr int ID = SYS_NSF2D, D = 2, M = 12, MC = 4;
    using Mms = Mms_nsf2d;
    struct Ctx { R u[2], du[2], ul[2], dp, tau[2][2], qh[2]; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R rho = P.ref[0] + dQ[0];
        const R r = R(1) / rho;
        R dke = R(0), u2 = R(0);
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            c.du[a] = (dQ[1 + a] - P.cst[a] * dQ[0]) * r;
            c.u[a] = P.cst[a] + c.du[a];
            c.ul[a] = c.u[a] * P.il;
            dke += dQ[1 + a] * c.u[a] + P.ref[1 + a] * c.du[a];
            u2 += c.u[a] * c.u[a];
        }
        const R gm1 = P.par[0] - R(1);
        c.dp = gm1 * (dQ[3] - R(0.5) * dke);
        const R T = (P.cst[3] + c.dp) * r;
        const R muL = P.par[1] * P.dL, KL = P.par[2] * P.dL;
        R gu[2][2], dT[2];
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            gu[0][b] = (dQ[6 + b] - c.u[0] * dQ[4 + b]) * r;
            gu[1][b] = (dQ[8 + b] - c.u[1] * dQ[4 + b]) * r;
            const R dpb = gm1 * (dQ[10 + b] - c.u[0] * dQ[6 + b] - c.u[1] * dQ[8 + b] + R(0.5) * u2 * dQ[4 + b]);
            dT[b] = (dpb - T * dQ[4 + b]) * r;
        }
        const R dv = R(2.0 / 3.0) * muL * (gu[0][0] + gu[1][1]);
        c.tau[0][0] = R(2) * muL * gu[0][0] - dv;
        c.tau[1][1] = R(2) * muL * gu[1][1] - dv;
        c.tau[0][1] = c.tau[1][0] = muL * (gu[0][1] + gu[1][0]);
#pragma unroll
        for (int j = 0; j < 2; ++j) c.qh[j] = c.tau[j][0] * c.u[0] + c.tau[j][1] * c.u[1] + KL * dT[j];
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2]; S = R(0);
        } else if constexpr (k <= 2) {
            constexpr int a = k - 1;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                R v = dQ[1 + a] * c.u[j] + P.ref[1 + a] * c.du[j];
                if (j == a) v += c.dp;
                F[j] = P.il * v - c.tau[a][j];
            }
            S = R(0);
        } else if constexpr (k == 3) {
#pragma unroll
            for (int j = 0; j < 2; ++j) F[j] = P.il * ((dQ[3] + c.dp) * c.u[j] + P.cst[4] * c.du[j]) - c.qh[j];
            S = R(0);
        } else {
            constexpr int v = (k - 4) / 2, b = (k - 4) % 2;
            F[0] = dQ[k] * c.ul[0]; F[1] = dQ[k] * c.ul[1];
            F[b] -= dQ[v] * P.inv_gtau;
            S = -dQ[k] * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double u = Q[1] / Q[0], v = Q[2] / Q[0];
        const double p = (P.par[0] - 1.0) * (Q[3] - 0.5 * Q[0] * (u * u + v * v));
        const double cc = sqrt(P.par[0] * p / Q[0]);
        out[0] = fmax(fabs(u), fabs(v)) + cc; out[1] = sqrt(u * u + v * v) + cc;
        out[2] = sqrt(fmax(4.0 * P.par[1] * P.dL / (3.0 * Q[0]), P.par[2] * P.dL * (P.par[0] - 1.0) / Q[0]) * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ NSF 3D
// eq (3.23), with derived-parent trackers after eq (3.27) (L495-L497):
// Q = (rho, m(3), E, G^L_ab = dx d_b u_a [index 5+3a+b], H^L_b = dx d_b T [index 14+b]), T = p/rho.
// par = {gamma, mu, K}.  Reference: rho0, E0 free; m0 = 0, trackers 0 (checked on the host).
//   sigma_ab = mu_L (G_ab + G_ba - 2/3 tr G delta_ab)
//   dF_rho,j = m_j/lam;  dF_ma,j = (m_a u_j + delta_aj dp)/lam - sigma_aj
//   dF_E,j = (E0 + p0 + dE + dp) u_j/lam - sigma_jb u_b - K_L H_j
//   dF_Gab,j = G_ab u_j/lam - delta_jb u_a/g_tau;  dF_Hb,j = H_b u_j/lam - delta_jb (T - T0)/g_tau
//   T - T0 = (dp - T0 drho)/rho;  s_G = -G/g_tau, s_H = -H/g_tau
template <class R> struct SysNsf3D {
    static constexpr int ID = SYS_NSF3D, D = 3, M = 17, MC = 5;
    using Mms = Mms_nsf3d;
    struct Ctx { R u[3], ul[3], dp, dT, sig[6], Hh; };   // ul = u/lambda; sig: xx yy zz xy xz yz
    __device__ __forceinline__ static int sidx(int a, int b) { return a == b ? a : (a + b + 2); }
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R rho = P.ref[0] + dQ[0];
        const R r = R(1) / rho;
        R ke = R(0);
        for (int a = 0; a < 3; ++a) { c.u[a] = dQ[1 + a] * r; c.ul[a] = c.u[a] * P.il; ke += dQ[1 + a] * c.u[a]; }
        c.dp = (P.par[0] - R(1)) * (dQ[4] - R(0.5) * ke);
        c.dT = (c.dp - P.cst[5] * dQ[0]) * r;
        const R muL = P.par[1] * P.dL;
        const R tr = (R(2.0 / 3.0) * muL) * (dQ[5] + dQ[9] + dQ[13]);
        c.sig[0] = R(2) * muL * dQ[5] - tr;
        c.sig[1] = R(2) * muL * dQ[9] - tr;
        c.sig[2] = R(2) * muL * dQ[13] - tr;
        c.sig[3] = muL * (dQ[5 + 1] + dQ[5 + 3]);    // xy
        c.sig[4] = muL * (dQ[5 + 2] + dQ[5 + 6]);    // xz
        c.sig[5] = muL * (dQ[5 + 5] + dQ[5 + 7]);    // yz
        c.Hh = P.cst[4] + dQ[4] + c.dp;              // E0 + p0 + dE + dp
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            for (int j = 0; j < 3; ++j) F[j] = P.il * dQ[1 + j];
            S = R(0);
        } else if constexpr (k <= 3) {
            constexpr int a = k - 1;
            for (int j = 0; j < 3; ++j) {
                R v = dQ[1 + a] * c.ul[j] - c.sig[sidx(a, j)];
                if (j == a) v += P.il * c.dp;
                F[j] = v;
            }
            S = R(0);
        } else if constexpr (k == 4) {
            const R KL = P.par[2] * P.dL;
            for (int j = 0; j < 3; ++j)
                F[j] = c.Hh * c.ul[j] - (c.sig[sidx(j, 0)] * c.u[0] + c.sig[sidx(j, 1)] * c.u[1] + c.sig[sidx(j, 2)] * c.u[2]) - KL * dQ[14 + j];
            S = R(0);
        } else if constexpr (k < 14) {
            constexpr int a = (k - 5) / 3, b = (k - 5) % 3;
            for (int j = 0; j < 3; ++j) F[j] = dQ[k] * c.ul[j];
            F[b] -= c.u[a] * P.inv_gtau;
            S = -dQ[k] * P.inv_gtau;
        } else {
            constexpr int b = k - 14;
            for (int j = 0; j < 3; ++j) F[j] = dQ[k] * c.ul[j];
            F[b] -= c.dT * P.inv_gtau;
            S = -dQ[k] * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double u[3] = {Q[1] / Q[0], Q[2] / Q[0], Q[3] / Q[0]};
        const double u2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
        const double p = (P.par[0] - 1.0) * (Q[4] - 0.5 * Q[0] * u2);
        const double cc = sqrt(P.par[0] * p / Q[0]);
        out[0] = fmax(fmax(fabs(u[0]), fabs(u[1])), fabs(u[2])) + cc;
        out[1] = sqrt(u2) + cc;
        const double kap = fmax(4.0 * P.par[1] * P.dL / (3.0 * Q[0]), P.par[2] * P.dL * (P.par[0] - 1.0) / Q[0]);
        out[2] = sqrt(kap * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ resistive MHD 3D
// eq (3.25), inviscid, no heat flux, no Powell source, current-density trackers
// J^L = dx curl B in place of the full grad B (C5).  Q = (rho, m(3), E, B(3), J^L(3)).
// par = {gamma, eta}.  Reference: rho0, E0 free; m0 = B0 = J0 = 0 (checked on the host).
//   p = (gamma-1)(E - rho|u|^2/2 - |B|^2/2),  p_tot = p + |B|^2/2
//   dF_ma,j = (m_a u_j - B_a B_j + delta_aj (dp + |B|^2/2))/lam
//   dF_E,j = ((E0 + p0 + dE + dp + |B|^2/2) u_j - B_j (u.B))/lam + eta_L (J x B)_j
//   dF_Bi,j = (B_i u_j - u_i B_j)/lam + eta_L eps_ijk J_k;   dF_Ji,j = J_i u_j/lam - eps_ijk B_k/g_tau
template <class R> struct SysMhd3D {
    static constexpr int ID = SYS_MHD3D, D = 3, M = 11, MC = 8;
    using Mms = void;
    struct Ctx { R u[3], ul[3], dpt, Hh, uB; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R rho = P.ref[0] + dQ[0];
        const R r = R(1) / rho;
        R ke = R(0), B2 = R(0);
        c.uB = R(0);
        for (int a = 0; a < 3; ++a) {
            c.u[a] = dQ[1 + a] * r; c.ul[a] = c.u[a] * P.il;
            ke += dQ[1 + a] * c.u[a]; B2 += dQ[5 + a] * dQ[5 + a]; c.uB += c.u[a] * dQ[5 + a];
        }
        const R dp = (P.par[0] - R(1)) * (dQ[4] - R(0.5) * ke - R(0.5) * B2);
        c.dpt = dp + R(0.5) * B2;
        c.Hh = P.cst[4] + dQ[4] + c.dpt;
    }
    // eps_ijk for (i, j): k index and sign; i != j
    __device__ __forceinline__ static constexpr int eps_k(int i, int j) { return 3 - i - j; }
    __device__ __forceinline__ static constexpr int eps_s(int i, int j) { return ((j - i + 3) % 3 == 1) ? +1 : -1; }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        const R* B = &dQ[5];
        const R* J = &dQ[8];
        S = R(0);
        if constexpr (k == 0) {
            for (int j = 0; j < 3; ++j) F[j] = P.il * dQ[1 + j];
        } else if constexpr (k <= 3) {
            constexpr int a = k - 1;
            for (int j = 0; j < 3; ++j) {
                R v = dQ[1 + a] * c.u[j] - B[a] * B[j];
                if (j == a) v += c.dpt;
                F[j] = P.il * v;
            }
        } else if constexpr (k == 4) {
            const R etaL = P.par[1] * P.dL;
            const R JxB[3] = {J[1] * B[2] - J[2] * B[1], J[2] * B[0] - J[0] * B[2], J[0] * B[1] - J[1] * B[0]};
            for (int j = 0; j < 3; ++j) F[j] = P.il * (c.Hh * c.u[j] - B[j] * c.uB) + etaL * JxB[j];
        } else if constexpr (k < 8) {
            constexpr int i = k - 5;
            const R etaL = P.par[1] * P.dL;
            for (int j = 0; j < 3; ++j) {
                if (j == i) { F[j] = R(0); continue; }                  // B_i u_i - u_i B_i = 0
                F[j] = P.il * (B[i] * c.u[j] - c.u[i] * B[j]) + R(eps_s(i, j)) * etaL * J[eps_k(i, j)];
            }
        } else {
            constexpr int i = k - 8;
            for (int j = 0; j < 3; ++j) {
                F[j] = J[i] * c.ul[j];
                if (j != i) F[j] -= R(eps_s(i, j)) * P.inv_gtau * B[eps_k(i, j)];
            }
            S = -J[i] * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double rho = Q[0];
        const double u[3] = {Q[1] / rho, Q[2] / rho, Q[3] / rho};
        const double u2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
        const double B2 = Q[5] * Q[5] + Q[6] * Q[6] + Q[7] * Q[7];
        const double p = (P.par[0] - 1.0) * (Q[4] - 0.5 * rho * u2 - 0.5 * B2);
        const double a2 = P.par[0] * p / rho, b2 = B2 / rho;
        double m0 = 0.0;
        for (int a = 0; a < 3; ++a) {
            const double ba2 = Q[5 + a] * Q[5 + a] / rho;
            const double cf = sqrt(0.5 * (a2 + b2 + sqrt(fmax((a2 + b2) * (a2 + b2) - 4.0 * a2 * ba2, 0.0))));
            m0 = fmax(m0, fabs(u[a]) + cf);
        }
        out[0] = m0;
        out[1] = sqrt(u2) + sqrt(a2 + b2);
        out[2] = sqrt(P.par[1] * P.dL * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ ultrarelativistic fluid
// eq (3.7)-(3.9): Q = (E, S_x, S_y), Phi_E = S, Phi_S = S (x) v + p I,
// p = (sqrt(D) - E)/3, D = 4E^2 - 3|S|^2, v = S/(E + p) = 3 S/W, W = 2E + sqrt(D); c = 1, no parameters.
// Delta form about (E0, S0): dD = 4 (2 E0 + dE) dE - 3 sum_a (2 S0a + dSa) dSa,  d sqrtD = dD/(sqrtD + sqrtD0),
// dp = (d sqrtD - dE)/3,  dW = 2 dE + d sqrtD,  dv_b = 3 (dS_b W0 - S0b dW)/(W W0),
// d(S_a v_b) = dS_a v_b + S0a dv_b.  With Q0 = 0 the reference constants vanish and this is the plain flux
// (sqrtD0 = W0 = 0 is handled by taking dv = v).
template <class R> struct SysUrf2D {
    static constexpr int ID = SYS_URF2D, D = 2, M = 3, MC = 3;
    using Mms = Mms_urf2d;
    struct Ctx { R v[2], dv[2], dp; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R E0 = P.ref[0], E = E0 + dQ[0];
        const R Sx = P.ref[1] + dQ[1], Sy = P.ref[2] + dQ[2];
        const R sD = sqrt(R(4) * E * E - R(3) * (Sx * Sx + Sy * Sy));
        const R W = R(2) * E + sD, iW = R(3) / W;
        c.v[0] = Sx * iW; c.v[1] = Sy * iW;
        const R sD0 = P.cst[2], W0 = P.cst[4];
        if (W0 != R(0)) {
            const R dD = R(4) * (R(2) * E0 + dQ[0]) * dQ[0] - R(3) * ((R(2) * P.ref[1] + dQ[1]) * dQ[1] + (R(2) * P.ref[2] + dQ[2]) * dQ[2]);
            const R dsD = dD / (sD + sD0);
            c.dp = (dsD - dQ[0]) * R(1.0 / 3.0);
            const R dW = R(2) * dQ[0] + dsD, k = iW / W0;
            c.dv[0] = (dQ[1] * W0 - P.ref[1] * dW) * k;
            c.dv[1] = (dQ[2] * W0 - P.ref[2] * dW) * k;
        } else {
            c.dp = (sD - E) * R(1.0 / 3.0);
            c.dv[0] = c.v[0]; c.dv[1] = c.v[1];
        }
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        S = R(0);
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2];
        } else {
            constexpr int a = k - 1;
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                R h = dQ[1 + a] * c.v[b] + P.ref[1 + a] * c.dv[b];
                if (a == b) h += c.dp;
                F[b] = P.il * h;
            }
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double cs2 = 1.0 / 3.0, cs = sqrt(cs2);
        const double p = (sqrt(4.0 * Q[0] * Q[0] - 3.0 * (Q[1] * Q[1] + Q[2] * Q[2])) - Q[0]) / 3.0;
        const double v[2] = {Q[1] / (Q[0] + p), Q[2] / (Q[0] + p)};
        const double v2 = v[0] * v[0] + v[1] * v[1];
        out[0] = 0.0;
        for (int a = 0; a < 2; ++a) {
            const double vn = fabs(v[a]);
            out[0] = fmax(out[0], (vn * (1.0 - cs2) + cs * sqrt(fmax((1.0 - v2) * (1.0 - v2 * cs2 - vn * vn * (1.0 - cs2)), 0.0))) / (1.0 - v2 * cs2));
        }
        const double vm = sqrt(v2);
        out[1] = (vm + cs) / (1.0 + vm * cs);
        out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ Maxwell TM
// eq (3.10)-(3.11): Q = (E_z, H_x, H_y), Phi = c ((-H_y, H_x), (0, E_z), (-E_z, 0)); par = {c}.
// Linear: the delta form is the flux itself.
template <class R> struct SysMaxwell2D {
    static constexpr int ID = SYS_MAXWELL2D, D = 2, M = 3, MC = 3;
    static constexpr bool LINEAR = true;
    using Mms = Mms_maxwell2d;
    struct Ctx {};
    __device__ __forceinline__ static void setup(Ctx&, const R (&)[M], const KParams<R>&) {}
    template <int k> __device__ __forceinline__ static void flux(const Ctx&, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        const R cl = P.par[0] * P.il;
        S = R(0);
        if constexpr (k == 0) { F[0] = -cl * dQ[2]; F[1] = cl * dQ[1]; }
        else if constexpr (k == 1) { F[0] = R(0); F[1] = cl * dQ[0]; }
        else { F[0] = -cl * dQ[0]; F[1] = R(0); }
    }
    __device__ static void wave(const double*, const KParams<double>& P, double* out) {
        out[0] = fabs(P.par[0]); out[1] = fabs(P.par[0]); out[2] = 0.0;    // eigenvalues {+c, -c, 0}
    }
};

// ------------------------------------------------------------------------------------------ shallow water over a bed
// eq (3.5)-(3.6): the SWE flux plus S = (0, -g h grad z_b); the static bed enters as the prescribed
// per-node field A = grad z_b (physical slope).  par = {g}; Q = (h, hu, hv)
template <class R> struct SysSwe2DBathy {
    static constexpr int ID = SYS_SWE2D_BATHY, D = 2, M = 3, MC = 3, NA = 2;
    using Mms = Mms_swe2d_bathy;
    struct Ctx { R u[2], du[2], dP, sl[2], gh; };
    __device__ __forceinline__ static void set_aux(Ctx& c, const R (&A)[NA]) { c.sl[0] = A[0]; c.sl[1] = A[1]; }
    __device__ __forceinline__ static void default_aux(Ctx& c) { c.sl[0] = R(0); c.sl[1] = R(0); }
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R h = P.ref[0] + dQ[0];
        const R rh = R(1) / h;
        for (int a = 0; a < 2; ++a) {
            c.du[a] = (dQ[1 + a] - P.cst[a] * dQ[0]) * rh;
            c.u[a] = P.cst[a] + c.du[a];
        }
        c.dP = R(0.5) * P.par[0] * dQ[0] * (R(2) * P.ref[0] + dQ[0]);
        c.gh = (P.dt * P.par[0]) * h;
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2];
            S = R(0);
        } else {
            constexpr int a = k - 1;
            for (int j = 0; j < 2; ++j) {
                R v = dQ[1 + a] * c.u[j] + P.ref[1 + a] * c.du[j];
                if (j == a) v += c.dP;
                F[j] = P.il * v;
            }
            S = -c.gh * c.sl[a];
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double cc = sqrt(P.par[0] * Q[0]), u = Q[1] / Q[0], v = Q[2] / Q[0];
        out[0] = fmax(fabs(u), fabs(v)) + cc; out[1] = sqrt(u * u + v * v) + cc; out[2] = 0.0;
    }
};

// ------------------------------------------------------------------------------------------ homogenized NSF 3D
// eq (3.27) and the state/flux/source vectors below it, PAPER.md:L486-L497 (listing SM4.12): prescribed
// porosity alpha(x,t) and solid velocity u_s(x,t) are per-node inputs A = (alpha, u_s0, u_s1, u_s2); reduced tracker
// basis D^L = dx sym grad u [5..10: 00 11 22 01 02 12], H^L = dx grad T [11..13], T = p/rho.
// par = {gamma, mu, kappa, eta_drag}.  Reference: rho0, E0 free; m0 = 0, trackers 0 (checked on the host).
//   tau_ab = alpha mu_L (2 D_ab - 2/3 tr D delta_ab)
//   dF_ma,j = (m_a u_j + delta_aj dp)/lam - tau_aj;  dF_E,j = (E0 + p0 + dE + dp) u_j/lam - tau_jb u_b - alpha kappa_L H_j
//   dF_Dab,j = D_ab u_j/lam - (delta_ja u_b + delta_jb u_a)/(2 g_tau);  dF_Hb,j = H_b u_j/lam - delta_jb (T - T0)/g_tau
//   s_ma = dt (1-alpha)/eta (rho u_s,a - m_a);  s_E = s_m . u;  s_D = -D/g_tau;  s_H = -H/g_tau
template <class R> struct SysHcnsf3D {
    static constexpr int ID = SYS_HCNSF3D, D = 3, M = 14, MC = 5, NA = 4;
    using Mms = void;
    struct Ctx { R al, us[3], u[3], ul[3], dp, dT, sig[6], Hh, sm[3], sE; };   // sig: xx yy zz xy xz yz (alpha included)
    __device__ __forceinline__ static int sidx(int a, int b) { return a == b ? a : (a + b + 2); }
    __device__ __forceinline__ static void set_aux(Ctx& c, const R (&A)[NA]) { c.al = A[0]; c.us[0] = A[1]; c.us[1] = A[2]; c.us[2] = A[3]; }
    __device__ __forceinline__ static void default_aux(Ctx& c) { c.al = R(1); c.us[0] = c.us[1] = c.us[2] = R(0); }
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R rho = P.ref[0] + dQ[0];
        const R r = R(1) / rho;
        R ke = R(0);
        for (int a = 0; a < 3; ++a) { c.u[a] = dQ[1 + a] * r; c.ul[a] = c.u[a] * P.il; ke += dQ[1 + a] * c.u[a]; }
        c.dp = (P.par[0] - R(1)) * (dQ[4] - R(0.5) * ke);
        c.dT = (c.dp - P.cst[5] * dQ[0]) * r;
        const R amu = c.al * (P.par[1] * P.dL);
        const R tr = (R(2.0 / 3.0) * amu) * (dQ[5] + dQ[6] + dQ[7]);
        for (int q = 0; q < 3; ++q) c.sig[q] = R(2) * amu * dQ[5 + q] - tr;
        for (int q = 3; q < 6; ++q) c.sig[q] = R(2) * amu * dQ[5 + q];
        c.Hh = P.cst[4] + dQ[4] + c.dp;
        const R drag = (R(1) - c.al) * (P.dt / P.par[3]);
        c.sE = R(0);
        for (int a = 0; a < 3; ++a) { c.sm[a] = drag * (rho * c.us[a] - dQ[1 + a]); c.sE += c.sm[a] * c.u[a]; }
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            for (int j = 0; j < 3; ++j) F[j] = P.il * dQ[1 + j];
            S = R(0);
        } else if constexpr (k <= 3) {
            constexpr int a = k - 1;
            for (int j = 0; j < 3; ++j) {
                R v = dQ[1 + a] * c.ul[j] - c.sig[sidx(a, j)];
                if (j == a) v += P.il * c.dp;
                F[j] = v;
            }
            S = c.sm[a];
        } else if constexpr (k == 4) {
            const R aK = c.al * (P.par[2] * P.dL);
            for (int j = 0; j < 3; ++j)
                F[j] = c.Hh * c.ul[j] - (c.sig[sidx(j, 0)] * c.u[0] + c.sig[sidx(j, 1)] * c.u[1] + c.sig[sidx(j, 2)] * c.u[2]) - aK * dQ[11 + j];
            S = c.sE;
        } else if constexpr (k < 11) {
            // D_ab: k = 5 + q, q -> (a, b) = (0,0) (1,1) (2,2) (0,1) (0,2) (1,2)
            constexpr int q = k - 5;
            constexpr int a = q < 3 ? q : (q == 5 ? 1 : 0), b = q < 3 ? q : (q == 3 ? 1 : 2);
            const R h = R(0.5) * P.inv_gtau;
            for (int j = 0; j < 3; ++j) F[j] = dQ[k] * c.ul[j];
            F[a] -= h * c.u[b];
            F[b] -= h * c.u[a];
            S = -dQ[k] * P.inv_gtau;
        } else {
            constexpr int b = k - 11;
            for (int j = 0; j < 3; ++j) F[j] = dQ[k] * c.ul[j];
            F[b] -= c.dT * P.inv_gtau;
            S = -dQ[k] * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double u[3] = {Q[1] / Q[0], Q[2] / Q[0], Q[3] / Q[0]};
        const double u2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
        const double p = (P.par[0] - 1.0) * (Q[4] - 0.5 * Q[0] * u2);
        const double cc = sqrt(P.par[0] * p / Q[0]);
        out[0] = fmax(fmax(fabs(u[0]), fabs(u[1])), fabs(u[2])) + cc;
        out[1] = sqrt(u2) + cc;
        const double kap = fmax(4.0 * P.par[1] * P.dL / (3.0 * Q[0]), P.par[2] * P.dL * (P.par[0] - 1.0) / Q[0]);   // alpha <= 1
        out[2] = sqrt(kap * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ resistive MHD 2D
// eq (3.25), PAPER.md:L469-L484 (listing SM4.11 garbled: vector form), cascade on the six conserved fields (N = 6 + 12):
// Q = (rho, m0, m1, E, B0, B1, G^L_{V,b} = dx d_b V [index 6 + 2 v + b], V = rho, m0, m1, E, B0, B1); par = {gamma, mu, K, eta}.
// Reference: (rho0, m0, E0, B0) free (moving, magnetised reference), trackers 0 (host-checked).  Chain rule as NSF 2D plus
//   d_b p = (gamma-1)(G_E,b - u.G_m,b + |u|^2/2 G_rho,b - B.G_B,b),  j_z = G_B1,0 - G_B0,1,  div B = G_B0,0 + G_B1,1.
// Delta forms (every term O(dQ)):  d(m_a u_j) = dm_a u_j + m0_a du_j;  d(B_a B_j) = dB_a B_j + B0_a dB_j;
//   d|B|^2 = (2 B0 + dB).dB;  dp = (gamma-1)(dE - d(m.u)/2 - d|B|^2/2);  dpt = dp + d|B|^2/2;
//   d((E+pt) u_j) = (dE + dpt) u_j + (E0 + pt0) du_j;  d(B_j (u.B)) = dB_j (u.B) + B0_j d(u.B),  d(u.B) = du.B + u0.dB.
// Powell source -(div B)(0, B, u.B, u), read off tr G_B: state-dependent, taken at the full state.
template <class R> struct SysMhd2D {
    static constexpr int ID = SYS_MHD2D, D = 2, M = 18, MC = 6;
    using Mms = Mms_mhd2d;
    struct Ctx { R u[2], du[2], ul[2], B[2], dp_t, tau[2][2], qh[2], uB, duB, Hh, divB; };
    __device__ __forceinline__ static void setup(Ctx& c, const R (&dQ)[M], const KParams<R>& P) {
        const R rho = P.ref[0] + dQ[0];
        const R r = R(1) / rho;
        R dke = R(0), u2 = R(0), dB2 = R(0);
        c.uB = R(0); c.duB = R(0);
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            c.du[a] = (dQ[1 + a] - P.cst[a] * dQ[0]) * r;
            c.u[a] = P.cst[a] + c.du[a];
            c.ul[a] = c.u[a] * P.il;
            c.B[a] = P.ref[4 + a] + dQ[4 + a];
            dke += dQ[1 + a] * c.u[a] + P.ref[1 + a] * c.du[a];
            u2 += c.u[a] * c.u[a];
            dB2 += (R(2) * P.ref[4 + a] + dQ[4 + a]) * dQ[4 + a];
            c.uB += c.u[a] * c.B[a];
            c.duB += c.du[a] * c.B[a] + P.cst[a] * dQ[4 + a];
        }
        const R gm1 = P.par[0] - R(1);
        const R dp = gm1 * (dQ[3] - R(0.5) * dke - R(0.5) * dB2);
        c.dp_t = dp + R(0.5) * dB2;
        c.Hh = dQ[3] + c.dp_t;
        const R T = (P.cst[3] + dp) * r;
        const R muL = P.par[1] * P.dL, KL = P.par[2] * P.dL, etaL = P.par[3] * P.dL;
        R gu[2][2], dT[2];
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            gu[0][b] = (dQ[8 + b] - c.u[0] * dQ[6 + b]) * r;
            gu[1][b] = (dQ[10 + b] - c.u[1] * dQ[6 + b]) * r;
            const R dpb = gm1 * (dQ[12 + b] - c.u[0] * dQ[8 + b] - c.u[1] * dQ[10 + b] + R(0.5) * u2 * dQ[6 + b]
                                 - c.B[0] * dQ[14 + b] - c.B[1] * dQ[16 + b]);
            dT[b] = (dpb - T * dQ[6 + b]) * r;
        }
        const R dv = R(2.0 / 3.0) * muL * (gu[0][0] + gu[1][1]);
        c.tau[0][0] = R(2) * muL * gu[0][0] - dv;
        c.tau[1][1] = R(2) * muL * gu[1][1] - dv;
        c.tau[0][1] = c.tau[1][0] = muL * (gu[0][1] + gu[1][0]);
        const R jz = dQ[16] - dQ[15];                     // G_B1,0 - G_B0,1
        const R ejxB[2] = {-etaL * jz * c.B[1], etaL * jz * c.B[0]};
#pragma unroll
        for (int j = 0; j < 2; ++j) c.qh[j] = c.tau[j][0] * c.u[0] + c.tau[j][1] * c.u[1] + KL * dT[j] - ejxB[j];
        c.divB = P.il * (dQ[14] + dQ[17]);
    }
    template <int k> __device__ __forceinline__ static void flux(const Ctx& c, const R (&dQ)[M], const KParams<R>& P, R (&F)[D], R& S) {
        if constexpr (k == 0) {
            F[0] = P.il * dQ[1]; F[1] = P.il * dQ[2]; S = R(0);
        } else if constexpr (k <= 2) {
            constexpr int a = k - 1;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                R v = dQ[1 + a] * c.u[j] + P.ref[1 + a] * c.du[j] - (dQ[4 + a] * c.B[j] + P.ref[4 + a] * dQ[4 + j]);
                if (j == a) v += c.dp_t;
                F[j] = P.il * v - c.tau[a][j];
            }
            S = -c.divB * c.B[a];
        } else if constexpr (k == 3) {
#pragma unroll
            for (int j = 0; j < 2; ++j)
                F[j] = P.il * (c.Hh * c.u[j] + P.cst[4] * c.du[j] - (dQ[4 + j] * c.uB + P.ref[4 + j] * c.duB)) - c.qh[j];
            S = -c.divB * c.uB;
        } else if constexpr (k <= 5) {
            constexpr int i = k - 4;
            const R etaL = P.par[3] * P.dL;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                // d(B_i u_j - u_i B_j) = dB_i u_j + B0_i du_j - du_i B_j - u0_i dB_j
                R v = R(0);
                if (j != i) v = dQ[4 + i] * c.u[j] + P.ref[4 + i] * c.du[j] - c.du[i] * c.B[j] - P.cst[i] * dQ[4 + j];
                F[j] = P.il * v - etaL * dQ[6 + 2 * (4 + i) + j];
            }
            S = -c.divB * c.u[i];
        } else {
            constexpr int v = (k - 6) / 2, b = (k - 6) % 2;
            F[0] = dQ[k] * c.ul[0]; F[1] = dQ[k] * c.ul[1];
            F[b] -= dQ[v] * P.inv_gtau;
            S = -dQ[k] * P.inv_gtau;
        }
    }
    __device__ static void wave(const double* Q, const KParams<double>& P, double* out) {
        const double rho = Q[0];
        const double u[2] = {Q[1] / rho, Q[2] / rho};
        const double u2 = u[0] * u[0] + u[1] * u[1];
        const double B2 = Q[4] * Q[4] + Q[5] * Q[5];
        const double p = (P.par[0] - 1.0) * (Q[3] - 0.5 * rho * u2 - 0.5 * B2);
        const double a2 = P.par[0] * p / rho, b2 = B2 / rho;
        double m0 = 0.0;
        for (int a = 0; a < 2; ++a) {
            const double ba2 = Q[4 + a] * Q[4 + a] / rho;
            const double cf = sqrt(0.5 * (a2 + b2 + sqrt(fmax((a2 + b2) * (a2 + b2) - 4.0 * a2 * ba2, 0.0))));
            m0 = fmax(m0, fabs(u[a]) + cf);
        }
        out[0] = m0;
        out[1] = sqrt(u2) + sqrt(a2 + b2);
        const double kap = fmax(fmax(4.0 * P.par[1] * P.dL / (3.0 * rho), P.par[2] * P.dL * (P.par[0] - 1.0) / rho), P.par[3] * P.dL);
        out[2] = sqrt(kap * P.inv_gtau);
    }
};

// ------------------------------------------------------------------------------------------ generated counterparts
// The plain lattice flux/source that gen/cascade.py DERIVES (Alg 2.1 Split/Cascade/Assemble/Emit) for the same system, where one
// is emitted: what lbmk_flux_selfcheck compares the hand-written delta form against.
// c4 with forcing: the populations of the last tracker component wait in shared memory (cp.async) instead of registers -- measured
// 2.42 ms/step against 2.46 (two components: 2.46, three: 2.47)
#ifndef LBMK_NSF3D_PARK
#define LBMK_NSF3D_PARK 1
#endif
template <> struct ParkCount<SysNsf3D<float>> { static constexpr int value = LBMK_NSF3D_PARK; };

template <template <class> class S> struct GenOf { using type = void; };
template <> struct GenOf<SysEuler2D> { using type = Gen_euler2d; };
template <> struct GenOf<SysSwe2DBathy> { using type = Gen_swe2d_bathy; };
template <> struct GenOf<SysAdr2D> { using type = Gen_adr2d; };
template <> struct GenOf<SysAllenCahn2D> { using type = Gen_allencahn2d; };
template <> struct GenOf<SysInse2D> { using type = Gen_inse2d; };
template <> struct GenOf<SysNsf2D> { using type = Gen_nsf2d; };
template <> struct GenOf<SysMhd2D> { using type = Gen_mhd2d; };
template <> struct GenOf<SysNsf3D> { using type = Gen_nsf3d; };
template <> struct GenOf<SysAdvection2D> { using type = Gen_advection2d; };
template <> struct GenOf<SysBurgers2D> { using type = Gen_burgers2d; };
template <> struct GenOf<SysSwe2D> { using type = Gen_swe2d; };
template <> struct GenOf<SysUrf2D> { using type = Gen_urf2d; };
template <> struct GenOf<SysMaxwell2D> { using type = Gen_maxwell2d; };
template <> struct GenOf<SysElasticity2D> { using type = Gen_elasticity2d; };
template <> struct GenOf<SysHcnsf3D> { using type = Gen_hcnsf3d; };
template <> struct GenOf<SysMhd3D> { using type = Gen_mhd3d; };

}  // namespace lbmk
