// oracle/lbm_oracle.cpp -- TEST INFRASTRUCTURE (CPU oracle). Not part of the product path.
//
// A plain, slow, fp64 implementation of the paper's collide-and-stream scheme, written step by
// step in the paper's order and notation (SURVEY.md §8(c) "Algorithm"):
//   0. init      f_k,i = w_i (U_k + c_i . F_k / c_s^2)                     eq (2.7); L718
//   1a. moments  U_k = sum_i f_k,i                                          eq (2.6)
//   1b. flux / source at the current moments; explicit (x,t) forcing at t_n + dt/2
//   1c. BGK      f' = f - omega_k (f - f_eq) + w_i s_k                      eq (2.11)
//   1d. stream   f_k,i(x + c_i, t+dt) = f'_k,i(x), periodic wrap            eq (2.11)
//   2. readback  U_k = sum_i f_k,i
// Two-lattice push, no blocking, no fusion, no reordering.  omega_k = 1/tau_k with
// tau_k = 1/2 + tau_R dt for conserved fields and omega = 1/(g_tau+1) for tracker
// fields.  Optional "shifted" storage f* = f - f_eq(Q0, F0) is eq (2.23)
// applied literally in fp64 (a cross-check of the identity, not a different scheme).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use this.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "jets.hpp"
#include "mms_fields.hpp"
#include "systems.hpp"

namespace orc {

// Table SM1. Direction order (free choice):
// 0 rest; 1:+x 2:-x 3:+y 4:-y 5:+z 6:-z.
struct Lattice {
    int D, Q;
    int c[7][3];
    double w[7];
    double cs2;
};
static Lattice make_lattice(int dim) {
    Lattice L;
    std::memset(&L, 0, sizeof(L));
    L.D = dim;
    L.Q = 2 * dim + 1;
    const double w0 = (dim == 2) ? 1.0 / 3.0 : 1.0 / 4.0;
    const double w1 = (dim == 2) ? 1.0 / 6.0 : 1.0 / 8.0;
    L.cs2 = (dim == 2) ? 1.0 / 3.0 : 1.0 / 4.0;
    L.w[0] = w0;
    for (int a = 0; a < dim; ++a) {
        L.c[1 + 2 * a][a] = +1;
        L.c[2 + 2 * a][a] = -1;
        L.w[1 + 2 * a] = w1;
        L.w[2 + 2 * a] = w1;
    }
    return L;
}

struct Spec {  // mirrored field by field in oracle/__init__.py (ctypes)
    int32_t system, nx, ny, nz;
    int32_t bc;        // 0 periodic, 1 Dirichlet-MMS frame
    int32_t shifted;   // 0 plain f, 1 store f* of eq (2.23)
    int32_t mms_id;    // 0 none
    int32_t n_threads; // 0 = OpenMP default
    int32_t ox, oy, oz; // coordinate origin in nodes: x_j = (j + ox) dx  (sub-box runs)
    int32_t pad_;
    double dx, lam, g_tau, t0;
    double par[16], mms_par[16];
    double tau_R[MAXM];  // per conserved component
    double omega[MAXM];  // >= 0 overrides the derived rate of component k (tests: omega = 0, 1)
    double U_ref[MAXM];  // Q0 for the shifted form
    int32_t collision;   // 0 BGK (eq 2.11, the operator the paper runs); 1 two-relaxation-time (PAPER.md:L154 names it; textbook form below)
    int32_t pad2_;
    double trt_magic;    // Lambda = (1/omega_plus - 1/2)(1/omega_minus - 1/2)
};

struct Grid {
    Spec s;
    Lattice L;
    SysInfo si;
    Scaling sc;
    int64_t n;       // nodes
    int64_t step;
    double omega[MAXM];
    double omega_plus[MAXM];   // TRT: rate of the symmetric parts; omega[] is then the rate of the antisymmetric (flux-carrying) parts
    double F_ref[MAXM * 3];
    std::vector<double> f, g;  // f[(k*Q + i)*n + node]
    std::vector<double> aux;   // prescribed coefficient fields aux[a*n + node] (n_aux per system; zeros until orc_set_aux)
    bool inited;
};

static inline int64_t node_index(const Grid& G, int x, int y, int z) { return ((int64_t)z * G.s.ny + y) * G.s.nx + x; }
static inline int wrap(int a, int n) { return ((a % n) + n) % n; }

// the prescribed coefficient fields of one node (nullptr-safe: systems without aux never read A)
static inline void node_aux(const Grid& G, int64_t nd, double* A) {
    for (int a = 0; a < G.si.n_aux; ++a) A[a] = G.aux[(int64_t)a * G.n + nd];
}

static void coords(const Grid& G, int x, int y, int z, double* X) {
    X[0] = (x + G.s.ox) * G.s.dx;
    X[1] = (y + G.s.oy) * G.s.dx;
    X[2] = (z + G.s.oz) * G.s.dx;
}

// eq (2.7); in shifted storage the stored value is f - f_eq(Q0, F0), eq (2.23)
static void equilibrium(const Grid& G, const double* U, const double* F, double* feq /*[m][Q]*/) {
    const Lattice& L = G.L;
    for (int k = 0; k < G.si.m_total; ++k)
        for (int i = 0; i < L.Q; ++i) {
            double cF = 0.0, cF0 = 0.0;
            for (int a = 0; a < L.D; ++a) { cF += L.c[i][a] * F[k * 3 + a]; cF0 += L.c[i][a] * G.F_ref[k * 3 + a]; }
            double v = L.w[i] * (U[k] + cF / L.cs2);
            if (G.s.shifted) v -= L.w[i] * (G.s.U_ref[k] + cF0 / L.cs2);
            feq[k * L.Q + i] = v;
        }
}

static bool is_frame(const Grid& G, int x, int y, int z) {
    if (x == 0 || x == G.s.nx - 1 || y == 0 || y == G.s.ny - 1) return true;
    if (G.L.D == 3 && (z == 0 || z == G.s.nz - 1)) return true;
    return false;
}

// Dirichlet-MMS (the paper defines no boundary operator):
// the outermost node layer is reset to f_eq(Q_exact(x_b, t)) before each step and before readback.
static void fill_frame(Grid& G, double t) {
    const int m = G.si.m_total, Q = G.L.Q;
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < G.s.nz; ++z)
        for (int y = 0; y < G.s.ny; ++y)
            for (int x = 0; x < G.s.nx; ++x) {
                if (!is_frame(G, x, y, z)) continue;
                double X[3];
                coords(G, x, y, z, X);
                J1 Qe[MAXM];
                exact_state(G.s.system, G.s.mms_id, G.sc, G.s.mms_par, t, X[0], X[1], X[2], Qe);
                double U[MAXM], F[MAXM * 3], S[MAXM], feq[MAXM * 7], A[8];
                for (int k = 0; k < m; ++k) U[k] = Qe[k].v;
                const int64_t nd = node_index(G, x, y, z);
                node_aux(G, nd, A);
                flux_source<double>(G.s.system, U, A, G.sc, F, S);
                equilibrium(G, U, F, feq);
                for (int q = 0; q < m * Q; ++q) G.f[(int64_t)q * G.n + nd] = feq[q];
            }
}

static void one_step(Grid& G) {
    const int m = G.si.m_total, Q = G.L.Q;
    const Lattice& L = G.L;
    const double t_n = G.s.t0 + G.step * G.sc.dt;
    if (G.s.bc == 1) fill_frame(G, t_n);
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < G.s.nz; ++z)
        for (int y = 0; y < G.s.ny; ++y)
            for (int x = 0; x < G.s.nx; ++x) {
                const int64_t nd = node_index(G, x, y, z);
                double U[MAXM], F[MAXM * 3], S[MAXM], feq[MAXM * 7], A[8];
                // 1a. zeroth moments, eq (2.6)
                for (int k = 0; k < m; ++k) {
                    double s = 0.0;
                    for (int i = 0; i < Q; ++i) s += G.f[(int64_t)(k * Q + i) * G.n + nd];
                    U[k] = G.s.shifted ? G.s.U_ref[k] + s : s;
                }
                // 1b. flux and state source at the current moments; explicit forcing at the midpoint
                node_aux(G, nd, A);     // prescribed coefficient fields as last set by orc_set_aux
                flux_source<double>(G.s.system, U, A, G.sc, F, S);
                if (G.s.mms_id != 0) {
                    double X[3], sm[MAXM];
                    coords(G, x, y, z, X);
                    if (mms_source(G.s.system, G.s.mms_id, G.sc, G.s.mms_par, t_n + 0.5 * G.sc.dt, X[0], X[1], X[2], sm))
                        for (int k = 0; k < m; ++k) S[k] += sm[k];
                }
                equilibrium(G, U, F, feq);
                // 1c + 1d. BGK relaxation with plain w_i-weighted source, then push to x + c_i
                for (int k = 0; k < m; ++k)
                    for (int i = 0; i < Q; ++i) {
                        const double fi = G.f[(int64_t)(k * Q + i) * G.n + nd];
                        double fpost = fi - G.omega[k] * (fi - feq[k * Q + i]) + L.w[i] * S[k];
                        if (G.s.collision != 0) {
                            // two-relaxation-time operator (textbook form; the paper names it at L154 as consuming the same
                            // equilibria): with ibar the direction opposite to i,  f+- = (f_i +- f_ibar)/2  and likewise f_eq+-,
                            //   f' = f_i - omega_plus (f+ - f_eq+) - omega_minus (f- - f_eq-) + w_i s_k .
                            // f_eq- = w_i c_i.F/c_s^2 carries the flux, so omega_minus = omega_k keeps the relaxation diffusion of
                            // eq (2.17); omega_plus follows from the magic parameter Lambda.
                            const int ib = (i == 0) ? 0 : (((i - 1) ^ 1) + 1);
                            const double fb = G.f[(int64_t)(k * Q + ib) * G.n + nd];
                            const double fp = 0.5 * (fi + fb), fm = 0.5 * (fi - fb);
                            const double ep = 0.5 * (feq[k * Q + i] + feq[k * Q + ib]), em = 0.5 * (feq[k * Q + i] - feq[k * Q + ib]);
                            fpost = fi - G.omega_plus[k] * (fp - ep) - G.omega[k] * (fm - em) + L.w[i] * S[k];
                        }
                        const int xd = wrap(x + L.c[i][0], G.s.nx), yd = wrap(y + L.c[i][1], G.s.ny), zd = wrap(z + L.c[i][2], G.s.nz);
                        G.g[(int64_t)(k * Q + i) * G.n + node_index(G, xd, yd, zd)] = fpost;
                    }
            }
    G.f.swap(G.g);
    G.step += 1;
}

}  // namespace orc

using namespace orc;

extern "C" {

int orc_system_info(int sys, int* m_conserved, int* m_total, int* dim, int* Q) {
    if (sys < 0 || sys >= SYS_COUNT) return 1;
    SysInfo si = sys_info(sys);
    *m_conserved = si.m_conserved; *m_total = si.m_total; *dim = si.dim; *Q = 2 * si.dim + 1;
    return 0;
}
int orc_system_n_aux(int sys) { return (sys < 0 || sys >= SYS_COUNT) ? -1 : sys_info(sys).n_aux; }

int orc_lattice(int dim, int* c /*[Q][3]*/, double* w /*[Q]*/, double* cs2) {
    if (dim != 2 && dim != 3) return 1;
    Lattice L = make_lattice(dim);
    for (int i = 0; i < L.Q; ++i) { w[i] = L.w[i]; for (int a = 0; a < 3; ++a) c[i * 3 + a] = L.c[i][a]; }
    *cs2 = L.cs2;
    return 0;
}

void* orc_create(const Spec* sp) {
    if (sp->system < 0 || sp->system >= SYS_COUNT) return nullptr;
    Grid* G = new Grid();
    G->s = *sp;
    G->si = sys_info(sp->system);
    G->L = make_lattice(G->si.dim);
    if (G->si.dim == 2 && sp->nz != 1) { delete G; return nullptr; }
    G->sc.par = G->s.par;
    G->sc.dx = sp->dx; G->sc.lam = sp->lam; G->sc.dt = sp->dx / sp->lam; G->sc.g_tau = sp->g_tau;
    G->n = (int64_t)sp->nx * sp->ny * sp->nz;
    G->step = 0;
    G->inited = false;
    for (int k = 0; k < G->si.m_total; ++k) {
        double om = (k < G->si.m_conserved) ? 1.0 / (0.5 + sp->tau_R[k] * G->sc.dt)   // tau_LB = 1/2 + tau_R dt, L194
                                            : 1.0 / (sp->g_tau + 1.0);                 // tracker rate, L718
        if (sp->omega[k] >= 0.0) om = sp->omega[k];
        G->omega[k] = om;
        // Lambda = (1/omega_plus - 1/2)(1/omega_minus - 1/2); omega_minus = 2 (no relaxation diffusion) leaves omega_plus free: 1
        const double tm = 1.0 / om - 0.5;
        G->omega_plus[k] = (sp->collision == 1 && om > 0.0) ? (tm > 0.0 ? 1.0 / (0.5 + sp->trt_magic / tm) : 1.0) : om;
        // collision 2, regularised: the non-equilibrium part is projected onto its first moment before relaxing,
        // f_neq,i -> w_i c_i.Pi/c_s^2, Pi = sum_j c_j (f_j - f_eq,j); on D2Q5 / D3Q7 that leaves the antisymmetric parts untouched and
        // removes the symmetric ones, i.e. it IS the two-rate form with omega_plus = 1 (pinned against the projection in tests/test_trt.py)
        if (sp->collision == 2) G->omega_plus[k] = 1.0;
    }
    {   // F0 = F(Q0) for the shifted storage, eq (2.23)
        double S[MAXM];
        for (int q = 0; q < MAXM * 3; ++q) G->F_ref[q] = 0.0;
        // prescribed fields at the reference state: alpha = 1 (pure fluid), everything else 0 (they multiply terms that
        // vanish at a uniform reference with zero trackers)
        double A0[8] = {1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        if (G->si.n_aux > 0 && sp->system != SYS_HCNSF3D) A0[0] = 0.0;
        if (sp->shifted) flux_source<double>(sp->system, G->s.U_ref, A0, G->sc, G->F_ref, S);
    }
    G->aux.assign((size_t)G->si.n_aux * G->n, 0.0);
    G->f.assign((size_t)G->si.m_total * G->L.Q * G->n, 0.0);
    G->g.assign((size_t)G->si.m_total * G->L.Q * G->n, 0.0);
#ifdef _OPENMP
    if (sp->n_threads > 0) omp_set_num_threads(sp->n_threads);
#endif
    return G;
}

void orc_destroy(void* h) { delete (Grid*)h; }

int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// step 0: all populations (conserved and tracker) at the equilibrium of U, eq (2.7)
int orc_init_from_U(void* h, const double* U_in /*[m][nz][ny][nx]*/) {
    Grid& G = *(Grid*)h;
    const int m = G.si.m_total, Q = G.L.Q;
#pragma omp parallel for schedule(static)
    for (int64_t nd = 0; nd < G.n; ++nd) {
        double U[MAXM], F[MAXM * 3], S[MAXM], feq[MAXM * 7], A[8];
        for (int k = 0; k < m; ++k) U[k] = U_in[(int64_t)k * G.n + nd];
        node_aux(G, nd, A);
        flux_source<double>(G.s.system, U, A, G.sc, F, S);
        equilibrium(G, U, F, feq);
        for (int q = 0; q < m * Q; ++q) G.f[(int64_t)q * G.n + nd] = feq[q];
    }
    G.step = 0;
    G.inited = true;
    return 0;
}

// prescribed coefficient fields A[a][nz][ny][nx] (bed slope of eq 3.5): used by every later flux/source
// evaluation until replaced (time-dependent fields: call again between steps)
int orc_set_aux(void* h, const double* A_in) {
    Grid& G = *(Grid*)h;
    if (G.si.n_aux == 0) return 1;
    std::memcpy(G.aux.data(), A_in, G.aux.size() * sizeof(double));
    return 0;
}

int orc_set_f(void* h, const double* f_in /*[m][Q][nz][ny][nx]*/) {
    Grid& G = *(Grid*)h;
    std::memcpy(G.f.data(), f_in, G.f.size() * sizeof(double));
    G.step = 0;
    G.inited = true;
    return 0;
}

int orc_step(void* h, int n_steps) {
    Grid& G = *(Grid*)h;
    if (!G.inited) return 2;
    for (int s = 0; s < n_steps; ++s) one_step(G);
    return 0;
}

int orc_read_f(void* h, double* f_out) {
    Grid& G = *(Grid*)h;
    std::memcpy(f_out, G.f.data(), G.f.size() * sizeof(double));
    return 0;
}

// step 2: U_k = sum_i f_k,i (+ Q0 in shifted storage)
int orc_read_U(void* h, double* U_out) {
    Grid& G = *(Grid*)h;
    const int m = G.si.m_total, Q = G.L.Q;
    if (G.s.bc == 1) fill_frame(G, G.s.t0 + G.step * G.sc.dt);
    for (int k = 0; k < m; ++k)
        for (int64_t nd = 0; nd < G.n; ++nd) {
            double s = 0.0;
            for (int i = 0; i < Q; ++i) s += G.f[(int64_t)(k * Q + i) * G.n + nd];
            U_out[(int64_t)k * G.n + nd] = G.s.shifted ? G.s.U_ref[k] + s : s;
        }
    return 0;
}

int orc_time(void* h, int64_t* step, double* t) {
    Grid& G = *(Grid*)h;
    *step = G.step;
    *t = G.s.t0 + G.step * G.sc.dt;
    return 0;
}

int orc_omega(void* h, double* omega_out) {
    Grid& G = *(Grid*)h;
    for (int k = 0; k < G.si.m_total; ++k) omega_out[k] = G.omega[k];
    return 0;
}
int orc_omega_plus(void* h, double* omega_out) {
    Grid& G = *(Grid*)h;
    for (int k = 0; k < G.si.m_total; ++k) omega_out[k] = G.omega_plus[k];
    return 0;
}

// exact augmented state on the grid at time t (trackers = dx * analytic gradient)
int orc_exact_U(void* h, double t, double* U_out) {
    Grid& G = *(Grid*)h;
    const int m = G.si.m_total;
    int ok = 0;
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < G.s.nz; ++z)
        for (int y = 0; y < G.s.ny; ++y)
            for (int x = 0; x < G.s.nx; ++x) {
                double X[3];
                coords(G, x, y, z, X);
                J1 Qe[MAXM];
                if (!exact_state(G.s.system, G.s.mms_id, G.sc, G.s.mms_par, t, X[0], X[1], X[2], Qe)) { ok = 1; continue; }
                for (int k = 0; k < m; ++k) U_out[(int64_t)k * G.n + node_index(G, x, y, z)] = Qe[k].v;
            }
    return ok;
}

// pointwise hooks for the pins ------------------------------------------------------------------
int orc_flux_source(void* h, const double* U, const double* A /*[n_aux] or NULL*/, double* F /*[m][3]*/, double* S /*[m]*/) {
    Grid& G = *(Grid*)h;
    double A0[8] = {0};
    flux_source<double>(G.s.system, U, A ? A : A0, G.sc, F, S);
    return 0;
}
int orc_equilibrium(void* h, const double* U, const double* F, double* feq /*[m][Q]*/) {
    Grid& G = *(Grid*)h;
    equilibrium(G, U, F, feq);
    return 0;
}
int orc_mms_source(void* h, double t, double x, double y, double z, double* s_out /*[m]*/) {
    Grid& G = *(Grid*)h;
    return mms_source(G.s.system, G.s.mms_id, G.sc, G.s.mms_par, t, x, y, z, s_out) ? 0 : 1;
}
int orc_exact_point(void* h, double t, double x, double y, double z, double* Q_out /*[m]*/) {
    Grid& G = *(Grid*)h;
    J1 Qe[MAXM];
    if (!exact_state(G.s.system, G.s.mms_id, G.sc, G.s.mms_par, t, x, y, z, Qe)) return 1;
    for (int k = 0; k < G.si.m_total; ++k) Q_out[k] = Qe[k].v;
    return 0;
}

// sub-characteristic check, eq (2.19)-(2.20): maxima over the grid, in LATTICE units
// out[0] per-axis, out[1] isotropic, out[2] tracker-parent diffusive signal speed
int orc_max_wave_speed(void* h, double* out3) {
    Grid& G = *(Grid*)h;
    const int m = G.si.m_total, Q = G.L.Q;
    double o0 = 0.0, o1 = 0.0, o2 = 0.0;
    for (int64_t nd = 0; nd < G.n; ++nd) {
        double U[MAXM], ws[3];
        for (int k = 0; k < m; ++k) {
            double s = 0.0;
            for (int i = 0; i < Q; ++i) s += G.f[(int64_t)(k * Q + i) * G.n + nd];
            U[k] = G.s.shifted ? G.s.U_ref[k] + s : s;
        }
        wave_speeds(G.s.system, U, G.sc, ws);
        o0 = std::fmax(o0, ws[0] / G.sc.lam);
        o1 = std::fmax(o1, ws[1] / G.sc.lam);
        o2 = std::fmax(o2, ws[2]);
    }
    out3[0] = o0; out3[1] = o1; out3[2] = o2;
    return 0;
}

// for every node x: linear index of the node whose post-collision population `dir` arrives at x,
// i.e. wrap(x - c_dir)  (SURVEY.md §8(c) "Canonical population state")
int orc_stream_index_map(void* h, int dir, int64_t* src_out) {
    Grid& G = *(Grid*)h;
    if (dir < 0 || dir >= G.L.Q) return 1;
    for (int z = 0; z < G.s.nz; ++z)
        for (int y = 0; y < G.s.ny; ++y)
            for (int x = 0; x < G.s.nx; ++x) {
                const int xs = wrap(x - G.L.c[dir][0], G.s.nx), ys = wrap(y - G.L.c[dir][1], G.s.ny), zs = wrap(z - G.L.c[dir][2], G.s.nz);
                src_out[node_index(G, x, y, z)] = node_index(G, xs, ys, zs);
            }
    return 0;
}

}  // extern "C"
