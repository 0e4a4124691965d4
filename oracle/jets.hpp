// oracle/jets.hpp -- TEST INFRASTRUCTURE (CPU oracle). Not part of the product path.
//
// Truncated Taylor "jets" in the four variables (t, x, y, z), used only to form the
// manufactured-solution forcing of eq (4.1), PAPER.md:L501-L502,
//     S_MMS(x,t) = d_t Q_exact + div Phi(Q_exact) - S(Q_exact),
// without writing any derivative by hand: exact primitives are written as functions of
// the coordinate jets, the conserved state and the flux are assembled with ordinary
// arithmetic, and the derivatives are read off the jet (product / quotient / chain rule).
//   J1: value + first derivatives (enough to take d_t Q and div Phi of an algebraic flux)
//   J2: value + first + second derivatives (needed where the exact tracker G = grad V is
//       itself a state component whose flux is differentiated once more)
// Shares no code with the CUDA path (whose forcing is a closed form emitted symbolically).
#pragma once
#include <cmath>

namespace orc {

constexpr int NV = 4;  // variable order: 0 = t, 1 = x, 2 = y, 3 = z

struct J1 {
    double v;
    double d[NV];
    J1() : v(0.0) { for (int i = 0; i < NV; ++i) d[i] = 0.0; }
    J1(double c) : v(c) { for (int i = 0; i < NV; ++i) d[i] = 0.0; }  // constant
};

inline J1 operator+(const J1& a, const J1& b) { J1 r; r.v = a.v + b.v; for (int i = 0; i < NV; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
inline J1 operator-(const J1& a, const J1& b) { J1 r; r.v = a.v - b.v; for (int i = 0; i < NV; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
inline J1 operator-(const J1& a) { J1 r; r.v = -a.v; for (int i = 0; i < NV; ++i) r.d[i] = -a.d[i]; return r; }
inline J1 operator*(const J1& a, const J1& b) {  // product rule
    J1 r; r.v = a.v * b.v; for (int i = 0; i < NV; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r;
}
inline J1 operator/(const J1& a, const J1& b) {  // quotient rule
    J1 r; r.v = a.v / b.v; for (int i = 0; i < NV; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v; return r;
}
inline J1 operator+(const J1& a, double c) { return a + J1(c); }
inline J1 operator+(double c, const J1& a) { return J1(c) + a; }
inline J1 operator-(const J1& a, double c) { return a - J1(c); }
inline J1 operator-(double c, const J1& a) { return J1(c) - a; }
inline J1 operator*(const J1& a, double c) { return a * J1(c); }
inline J1 operator*(double c, const J1& a) { return J1(c) * a; }
inline J1 operator/(const J1& a, double c) { return a / J1(c); }
inline J1 operator/(double c, const J1& a) { return J1(c) / a; }
inline J1 log(const J1& a) { J1 r; r.v = std::log(a.v); for (int i = 0; i < NV; ++i) r.d[i] = a.d[i] / a.v; return r; }
inline J1 sqrt(const J1& a) { J1 r; r.v = std::sqrt(a.v); for (int i = 0; i < NV; ++i) r.d[i] = a.d[i] / (2.0 * r.v); return r; }

struct J2 {
    double v;
    double d[NV];
    double h[NV][NV];  // full symmetric Hessian
    J2() : v(0.0) { for (int i = 0; i < NV; ++i) { d[i] = 0.0; for (int j = 0; j < NV; ++j) h[i][j] = 0.0; } }
    J2(double c) : J2() { v = c; }
    static J2 variable(int which, double value) { J2 r(value); r.d[which] = 1.0; return r; }
};

inline J2 operator+(const J2& a, const J2& b) {
    J2 r; r.v = a.v + b.v;
    for (int i = 0; i < NV; ++i) { r.d[i] = a.d[i] + b.d[i]; for (int j = 0; j < NV; ++j) r.h[i][j] = a.h[i][j] + b.h[i][j]; }
    return r;
}
inline J2 operator-(const J2& a) {
    J2 r; r.v = -a.v;
    for (int i = 0; i < NV; ++i) { r.d[i] = -a.d[i]; for (int j = 0; j < NV; ++j) r.h[i][j] = -a.h[i][j]; }
    return r;
}
inline J2 operator-(const J2& a, const J2& b) { return a + (-b); }
inline J2 operator*(const J2& a, const J2& b) {  // Leibniz to second order
    J2 r; r.v = a.v * b.v;
    for (int i = 0; i < NV; ++i) {
        r.d[i] = a.d[i] * b.v + a.v * b.d[i];
        for (int j = 0; j < NV; ++j)
            r.h[i][j] = a.h[i][j] * b.v + a.d[i] * b.d[j] + a.d[j] * b.d[i] + a.v * b.h[i][j];
    }
    return r;
}
// g(a) for a scalar function with g(a.v) = g0, g' = g1, g'' = g2 (chain rule)
inline J2 chain(const J2& a, double g0, double g1, double g2) {
    J2 r; r.v = g0;
    for (int i = 0; i < NV; ++i) {
        r.d[i] = g1 * a.d[i];
        for (int j = 0; j < NV; ++j) r.h[i][j] = g1 * a.h[i][j] + g2 * a.d[i] * a.d[j];
    }
    return r;
}
inline J2 sin(const J2& a) { return chain(a, std::sin(a.v), std::cos(a.v), -std::sin(a.v)); }
inline J2 cos(const J2& a) { return chain(a, std::cos(a.v), -std::sin(a.v), -std::cos(a.v)); }
inline J2 exp(const J2& a) { double e = std::exp(a.v); return chain(a, e, e, e); }
inline J2 recip(const J2& a) { double r = 1.0 / a.v; return chain(a, r, -r * r, 2.0 * r * r * r); }
inline J2 operator/(const J2& a, const J2& b) { return a * recip(b); }
inline J2 operator+(const J2& a, double c) { return a + J2(c); }
inline J2 operator+(double c, const J2& a) { return J2(c) + a; }
inline J2 operator-(const J2& a, double c) { return a - J2(c); }
inline J2 operator-(double c, const J2& a) { return J2(c) - a; }
inline J2 operator*(const J2& a, double c) { return a * J2(c); }
inline J2 operator*(double c, const J2& a) { return J2(c) * a; }
inline J2 operator/(const J2& a, double c) { return a * J2(1.0 / c); }

// value + first derivatives of a J2
inline J1 lower(const J2& a) { J1 r; r.v = a.v; for (int i = 0; i < NV; ++i) r.d[i] = a.d[i]; return r; }
// the jet of d a / d (variable `which`)
inline J1 diff(const J2& a, int which) { J1 r; r.v = a.d[which]; for (int i = 0; i < NV; ++i) r.d[i] = a.h[which][i]; return r; }

}  // namespace orc
