// lbmk_api.cu -- the C-ABI of include/lbmk.h: handles, validation, workspace layout, host-side grid scaling
// and the a-priori sub-characteristic check.  All arithmetic of the method runs in the kernels
// (kernels.cuh, systems.cuh); this file only derives launch parameters on the host:
//   dt = dx/lambda, omega_k = 1/(1/2 + tau_R,k dt) for conserved fields, omega = 1/(g_tau+1)
//   for tracker fields, the reference constants of the delta forms (systems.cuh header).
#include "../../include/lbmk.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "api_kernels.cuh"
#include "cascade_generated.cuh"
#include "ops.h"

using namespace lbmk;

struct lbmk_system {
    int id, lattice;
    double par[LBMK_MAX_PARAMS];
    int n_par;
    double tau_R[LBMK_MAX_COMPONENTS];
    double g_tau;
    double omega[LBMK_MAX_COMPONENTS];
    bool omega_set;
    double ref[LBMK_MAX_COMPONENTS];
    int mms_id;
    double mp[LBMK_MAX_PARAMS];
    double s_max;
    int collision;
    double trt_magic;
};

struct lbmk_grid {
    lbmk_system sys;
    const SysOps* ops;
    GridCore c;
    int precision;                 // lbmk_precision as given
    double dx, lam;
    long long opt_pattern, opt_kernel;
    bool bound, inited;
    size_t ws_bytes;
    size_t off_f[2], off_tab[3], off_coef, off_feq0, off_red, off_aux;
    long long opt_stepping;
    cudaEvent_t ev_boundary, ev_join;
    std::string err;
    cudaEvent_t ev0, ev1;
    bool have_events, timed;
};

static thread_local std::string g_sys_err;

static const SysOps* ops_of(int id) {
    switch (id) {
        case LBMK_SYS_ADVECTION2D: return ops_advection2d();
        case LBMK_SYS_BURGERS2D: return ops_burgers2d();
        case LBMK_SYS_SWE2D: return ops_swe2d();
        case LBMK_SYS_EULER2D: return ops_euler2d();
        case LBMK_SYS_ADR2D: return ops_adr2d();
        case LBMK_SYS_NSF3D_GRADTRACK: return ops_nsf3d();
        case LBMK_SYS_MHD3D_JTRACK: return ops_mhd3d();
        case LBMK_SYS_URF2D: return ops_urf2d();
        case LBMK_SYS_MAXWELL2D: return ops_maxwell2d();
        case LBMK_SYS_ALLENCAHN2D: return ops_allencahn2d();
        case LBMK_SYS_INSE2D: return ops_inse2d();
        case LBMK_SYS_ELASTICITY2D: return ops_elasticity2d();
        case LBMK_SYS_NSF2D_GRADTRACK: return ops_nsf2d();
        case LBMK_SYS_SWE2D_BATHY: return ops_swe2d_bathy();
        case LBMK_SYS_HCNSF3D: return ops_hcnsf3d();
        case LBMK_SYS_MHD2D: return ops_mhd2d();
    }
    return nullptr;
}
static const int N_PARAMS[LBMK_SYS_COUNT] = {2, 0, 1, 1, 4, 3, 2, 0, 1, 2, 2, 3, 3, 1, 4, 4};
static const int N_MMS_PARAMS[LBMK_SYS_COUNT] = {0, 1, 3, 0, 0, 4, 0, 0, 0, 0, 2, 0, 0, 6, 0, 0};

static lbmk_status sys_fail(lbmk_status s, const char* msg) { g_sys_err = msg; return s; }
static lbmk_status fail(lbmk_grid* g, lbmk_status s, const std::string& msg) { if (g) g->err = msg; else g_sys_err = msg; return s; }
static lbmk_status cuda_fail(lbmk_grid* g, cudaError_t e, const char* where) {
    return fail(g, LBMK_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CK(g, call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail((g), e_, (where)); } while (0)

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// evaluation of one emitted system (gen/cascade.py -> cascade_generated.cuh) on the host
template <class Gen>
static void gen_eval(const double* U, const double* A, const GenArgs<double>& ga, double* F3, double* S) {
    double F[LBMK_MAX_COMPONENTS * 3], A0[8] = {0};
    Gen::template flux<double>(U, A ? A : A0, ga, F, S);
    for (int k = 0; k < Gen::M; ++k)
        for (int a = 0; a < 3; ++a) F3[k * 3 + a] = a < Gen::D ? F[k * Gen::D + a] : 0.0;
}

extern "C" {

const char* lbmk_version(void) { return "lbmk 0.1 (sm_100a)"; }

const char* lbmk_last_error(const lbmk_grid* g) { return g ? g->err.c_str() : g_sys_err.c_str(); }

lbmk_status lbmk_lattice_constants(lbmk_lattice lattice, int* c, double* w, double* cs2) {
    if (lattice != LBMK_D2Q5 && lattice != LBMK_D3Q7) return sys_fail(LBMK_EINVAL, "unknown lattice");
    const int D = lattice == LBMK_D2Q5 ? 2 : 3, Q = 2 * D + 1;
    for (int i = 0; i < Q; ++i) {
        if (c) for (int a = 0; a < 3; ++a) c[i * 3 + a] = cvel(i, a);
        if (w) w[i] = (i == 0) ? (D == 2 ? Lattice<2>::w0 : Lattice<3>::w0) : (D == 2 ? Lattice<2>::w1 : Lattice<3>::w1);
    }
    if (cs2) *cs2 = D == 2 ? Lattice<2>::cs2 : Lattice<3>::cs2;
    return LBMK_OK;
}

// ------------------------------------------------------------------------------------------------ system
lbmk_status lbmk_system_create(lbmk_system_id id, lbmk_lattice lattice, const double* params, int n_params, lbmk_system** out) {
    if (!out) return sys_fail(LBMK_EINVAL, "out is NULL");
    *out = nullptr;
    const SysOps* ops = ops_of((int)id);
    if (!ops) return sys_fail(LBMK_EINVAL, "unknown system id");
    if ((ops->D == 2 && lattice != LBMK_D2Q5) || (ops->D == 3 && lattice != LBMK_D3Q7))
        return sys_fail(LBMK_EINVAL, "lattice does not match the system's dimension (2D: D2Q5, 3D: D3Q7)");
    if (n_params != N_PARAMS[id] || (n_params > 0 && !params)) return sys_fail(LBMK_EINVAL, "wrong number of system parameters");
    lbmk_system* s = new (std::nothrow) lbmk_system();
    if (!s) return sys_fail(LBMK_ENOMEM, "host allocation failed");
    memset(s, 0, sizeof(*s));
    s->id = id; s->lattice = lattice; s->n_par = n_params;
    for (int i = 0; i < n_params; ++i) s->par[i] = params[i];
    s->g_tau = 1.0;
    *out = s;
    return LBMK_OK;
}

lbmk_status lbmk_system_info(const lbmk_system* sys, int* m_conserved, int* m_total, int* dim, int* Q) {
    if (!sys) return sys_fail(LBMK_EINVAL, "sys is NULL");
    const SysOps* o = ops_of(sys->id);
    if (m_conserved) *m_conserved = o->MC;
    if (m_total) *m_total = o->M;
    if (dim) *dim = o->D;
    if (Q) *Q = 2 * o->D + 1;
    return LBMK_OK;
}

lbmk_status lbmk_system_aux_count(const lbmk_system* sys, int* n_aux) {
    if (!sys || !n_aux) return sys_fail(LBMK_EINVAL, "NULL argument");
    *n_aux = ops_of(sys->id)->n_aux;
    return LBMK_OK;
}

lbmk_status lbmk_system_set_relaxation(lbmk_system* sys, const double* tau_R, int n, double g_tau) {
    if (!sys || !tau_R) return sys_fail(LBMK_EINVAL, "NULL argument");
    const SysOps* o = ops_of(sys->id);
    if (n != 1 && n != o->MC) return sys_fail(LBMK_EINVAL, "tau_R: n must be 1 or m_conserved");
    for (int k = 0; k < o->MC; ++k) {
        sys->tau_R[k] = tau_R[n == 1 ? 0 : k];
        if (!(sys->tau_R[k] >= 0.0)) return sys_fail(LBMK_EINVAL, "tau_R must be >= 0");
    }
    if (o->M > o->MC && !(g_tau > 0.0)) return sys_fail(LBMK_EINVAL, "g_tau must be > 0 for tracker systems");
    sys->g_tau = g_tau > 0.0 ? g_tau : 1.0;
    return LBMK_OK;
}

lbmk_status lbmk_system_set_omega(lbmk_system* sys, const double* omega, int n) {
    if (!sys || !omega) return sys_fail(LBMK_EINVAL, "NULL argument");
    const SysOps* o = ops_of(sys->id);
    if (n != 1 && n != o->M) return sys_fail(LBMK_EINVAL, "omega: n must be 1 or m_total");
    for (int k = 0; k < o->M; ++k) {
        sys->omega[k] = omega[n == 1 ? 0 : k];
        if (!(sys->omega[k] >= 0.0 && sys->omega[k] <= 2.0)) return sys_fail(LBMK_EINVAL, "omega must lie in [0, 2]");
    }
    sys->omega_set = true;
    return LBMK_OK;
}

lbmk_status lbmk_system_set_reference(lbmk_system* sys, const double* U0, int n) {
    if (!sys || !U0) return sys_fail(LBMK_EINVAL, "NULL argument");
    const SysOps* o = ops_of(sys->id);
    if (n != o->M) return sys_fail(LBMK_EINVAL, "reference: n must be m_total");
    if (sys->id == LBMK_SYS_NSF3D_GRADTRACK || sys->id == LBMK_SYS_MHD3D_JTRACK || sys->id == LBMK_SYS_HCNSF3D) {
        for (int k = 0; k < n; ++k)
            if (k != 0 && k != 4 && U0[k] != 0.0)
                return sys_fail(LBMK_EUNSUPPORTED, "NSF3D/MHD3D/HCNSF3D delta forms need zero reference momentum, field and trackers");
    }
    if (sys->id == LBMK_SYS_MHD2D) {
        for (int k = 6; k < n; ++k)
            if (U0[k] != 0.0) return sys_fail(LBMK_EUNSUPPORTED, "MHD2D needs zero reference trackers");
    }
    if (sys->id == LBMK_SYS_ELASTICITY2D) {
        const double rest[6] = {1, 0, 0, 1, 0, 0};
        bool zero = true, is_rest = true;
        for (int k = 0; k < 6; ++k) { zero = zero && U0[k] == 0.0; is_rest = is_rest && U0[k] == rest[k]; }
        if (!zero && !is_rest) return sys_fail(LBMK_EUNSUPPORTED, "ELASTICITY2D reference state must be the rest configuration F = I, v = 0");
    }
    if (sys->id == LBMK_SYS_NSF2D_GRADTRACK) {
        for (int k = 4; k < n; ++k)
            if (U0[k] != 0.0) return sys_fail(LBMK_EUNSUPPORTED, "NSF2D needs zero reference trackers");
    }
    if (sys->id == LBMK_SYS_INSE2D) {
        for (int k = 1; k < n; ++k)
            if (U0[k] != 0.0) return sys_fail(LBMK_EUNSUPPORTED, "INSE2D delta form needs zero reference momentum and trackers");
    }
    if ((sys->id == LBMK_SYS_ADR2D || sys->id == LBMK_SYS_ALLENCAHN2D) && (U0[1] != 0.0 || U0[2] != 0.0))
        return sys_fail(LBMK_EUNSUPPORTED, "ADR2D needs zero reference trackers");
    for (int k = 0; k < n; ++k) sys->ref[k] = U0[k];
    return LBMK_OK;
}

lbmk_status lbmk_system_set_mms(lbmk_system* sys, int mms_id, const double* mms_params, int n) {
    if (!sys) return sys_fail(LBMK_EINVAL, "sys is NULL");
    if (mms_id == 0) { sys->mms_id = 0; return LBMK_OK; }
    const SysOps* o = ops_of(sys->id);
    if (mms_id != 1 || !o->has_mms) return sys_fail(LBMK_EUNSUPPORTED, "no manufactured solution compiled in for this (system, mms_id)");
    if (n != N_MMS_PARAMS[sys->id] || (n > 0 && !mms_params)) return sys_fail(LBMK_EINVAL, "wrong number of mms parameters");
    for (int i = 0; i < n; ++i) sys->mp[i] = mms_params[i];
    sys->mms_id = 1;
    return LBMK_OK;
}

lbmk_status lbmk_system_set_collision(lbmk_system* sys, int collision, double magic) {
    if (!sys) return sys_fail(LBMK_EINVAL, "sys is NULL");
    if (collision != LBMK_COLLISION_BGK && collision != LBMK_COLLISION_TRT && collision != LBMK_COLLISION_REGULARIZED)
        return sys_fail(LBMK_EINVAL, "unknown collision operator");
    if (collision == LBMK_COLLISION_TRT && !(magic > 0.0)) return sys_fail(LBMK_EINVAL, "TRT magic parameter must be > 0");
    sys->collision = collision;
    sys->trt_magic = magic;
    return LBMK_OK;
}

lbmk_status lbmk_system_set_wave_speed_bound(lbmk_system* sys, double s_max) {
    if (!sys || !(s_max >= 0.0)) return sys_fail(LBMK_EINVAL, "bad argument");
    sys->s_max = s_max;
    return LBMK_OK;
}

void lbmk_system_destroy(lbmk_system* sys) { delete sys; }

// ------------------------------------------------------------------------------------------------ grid
static bool is_shifted(int precision) { return precision == LBMK_F32_SHIFTED || precision == LBMK_F64_SHIFTED; }

// host-side derivation of the kernel parameter block (grid scaling + reference constants of the delta forms)
static void derive_params(lbmk_grid* g) {
    const lbmk_system& s = g->sys;
    const SysOps* o = g->ops;
    GridCore& c = g->c;
    KParams<double>& P = c.Pd;
    memset(&P, 0, sizeof(P));
    const double dt = g->dx / g->lam;
    c.dt = dt;
    P.nx = c.nx; P.ny = c.ny; P.nz = c.nz; P.n = c.n;
    P.il = 1.0 / g->lam;
    P.dL = dt / (g->dx * g->dx);
    P.inv_gtau = 1.0 / s.g_tau;
    P.dt = dt;
    for (int k = 0; k < o->M; ++k) {
        double om = (k < o->MC) ? 1.0 / (0.5 + s.tau_R[k] * dt)     // tau_LB = 1/2 + tau_R dt
                                : 1.0 / (s.g_tau + 1.0);            // tracker rate
        if (s.omega_set) om = s.omega[k];
        P.omega[k] = om;
        // TRT: Lambda = (1/omega_p - 1/2)(1/omega - 1/2); omega = 2 leaves omega_p free (1); omega = 0 (no collision) keeps 0
        const double tm = om > 0.0 ? 1.0 / om - 0.5 : 0.0;
        P.omega_p[k] = (s.collision == LBMK_COLLISION_TRT && om > 0.0) ? (tm > 0.0 ? 1.0 / (0.5 + s.trt_magic / tm) : 1.0) : om;
        if (s.collision == LBMK_COLLISION_REGULARIZED) P.omega_p[k] = 1.0;     // projection of f_neq onto its first moment = symmetric parts fully relaxed
        P.ref[k] = is_shifted(g->precision) ? s.ref[k] : 0.0;
    }
    for (int i = 0; i < 8; ++i) P.par[i] = s.par[i];
    const double* r = P.ref;
    switch (s.id) {
        case LBMK_SYS_SWE2D_BATHY:
        case LBMK_SYS_SWE2D:
            for (int a = 0; a < 2; ++a) P.cst[a] = r[0] != 0.0 ? r[1 + a] / r[0] : 0.0;
            break;
        case LBMK_SYS_NSF2D_GRADTRACK:
        case LBMK_SYS_EULER2D: {
            double ke = 0.0;
            for (int a = 0; a < 2; ++a) { P.cst[a] = r[0] != 0.0 ? r[1 + a] / r[0] : 0.0; ke += r[1 + a] * P.cst[a]; }
            P.cst[3] = (s.par[0] - 1.0) * (r[3] - 0.5 * ke);
            P.cst[4] = r[3] + P.cst[3];
        } break;
        case LBMK_SYS_URF2D: {
            const double D0 = 4.0 * r[0] * r[0] - 3.0 * (r[1] * r[1] + r[2] * r[2]);
            P.cst[2] = D0 > 0.0 ? std::sqrt(D0) : 0.0;
            P.cst[4] = 2.0 * r[0] + P.cst[2];
            P.cst[3] = (P.cst[2] - r[0]) / 3.0;
            for (int a = 0; a < 2; ++a) P.cst[a] = P.cst[4] != 0.0 ? 3.0 * r[1 + a] / P.cst[4] : 0.0;
        } break;
        case LBMK_SYS_MHD2D: {
            // u0 = m0/rho0; gas pressure p0 = (gamma-1)(E0 - m0.u0/2 - |B0|^2/2); cst[4] = E0 + p0 + |B0|^2/2
            double ke = 0.0;
            const double B2 = r[4] * r[4] + r[5] * r[5];
            for (int a = 0; a < 2; ++a) { P.cst[a] = r[0] != 0.0 ? r[1 + a] / r[0] : 0.0; ke += r[1 + a] * P.cst[a]; }
            P.cst[3] = (s.par[0] - 1.0) * (r[3] - 0.5 * ke - 0.5 * B2);
            P.cst[4] = r[3] + P.cst[3] + 0.5 * B2;
        } break;
        case LBMK_SYS_HCNSF3D:
        case LBMK_SYS_NSF3D_GRADTRACK:
        case LBMK_SYS_MHD3D_JTRACK:
            P.cst[3] = (s.par[0] - 1.0) * r[4];
            P.cst[4] = r[4] + P.cst[3];
            P.cst[5] = r[0] != 0.0 ? P.cst[3] / r[0] : 0.0;
            break;
        default: break;
    }
    MmsHostArgs& mh = c.mh;
    memset(&mh, 0, sizeof(mh));
    for (int i = 0; i < 16; ++i) { mh.par[i] = s.par[i]; mh.mp[i] = s.mp[i]; }
    mh.dx = g->dx; mh.dt = dt; mh.il = P.il; mh.gtau = s.g_tau;
    for (int i = 0; i < 8; ++i) { P.mms.par[i] = s.par[i]; P.mms.mp[i] = s.mp[i]; }
    P.mms.dx = g->dx; P.mms.dt = dt; P.mms.il = P.il; P.mms.gtau = s.g_tau;
    // fp32 image
    KParams<float>& F = c.Pf;
    memset(&F, 0, sizeof(F));
    F.nx = P.nx; F.ny = P.ny; F.nz = P.nz; F.n = P.n;
    for (int k = 0; k < MAXM; ++k) { F.omega[k] = (float)P.omega[k]; F.omega_p[k] = (float)P.omega_p[k]; F.ref[k] = (float)P.ref[k]; }
    for (int i = 0; i < 8; ++i) { F.par[i] = (float)P.par[i]; F.cst[i] = (float)P.cst[i]; F.mms.par[i] = (float)P.mms.par[i]; F.mms.mp[i] = (float)P.mms.mp[i]; }
    F.il = (float)P.il; F.dL = (float)P.dL; F.inv_gtau = (float)P.inv_gtau; F.dt = (float)P.dt;
    F.mms.dx = (float)P.mms.dx; F.mms.dt = (float)P.mms.dt; F.mms.il = (float)P.mms.il; F.mms.gtau = (float)P.mms.gtau;
}

static void resolve_options(lbmk_grid* g) {
    GridCore& c = g->c;
    c.pattern = g->opt_pattern == LBMK_PATTERN_AUTO ? (g->opt_stepping == LBMK_STEPPING_RESIDENT ? PATTERN_AA : PATTERN_PULL2) : (int)g->opt_pattern;
    if (c.bc == LBMK_DIRICHLET_MMS) c.pattern = PATTERN_PULL2;      // the frame refill needs canonical storage
    c.kernel = g->opt_kernel == LBMK_KERNEL_AUTO ? KERNEL_NODE : (int)g->opt_kernel;
    c.collision = g->sys.collision != LBMK_COLLISION_BGK ? 1 : 0;          // TRT and regularised share the two-rate kernel
    if (c.collision != 0) { c.pattern = PATTERN_PULL2; c.kernel = KERNEL_NODE; }   // the variants TRT is compiled for
    if (c.kernel == KERNEL_ROW && !g->ops->row_kernel_supported(c)) c.kernel = KERNEL_NODE;
    // Stepping: grids whose two population copies fit in L2 are launch-latency bound, not bandwidth bound (c1: 0.3 MB,
    // c2: 63 MB against 126 MB of L2) -> one cooperative launch per batch of steps; larger grids: one launch per step.
    const size_t esz = c.prec == PREC_F64 ? 8 : 4;
    const size_t state2 = 2 * (size_t)g->ops->M * (2 * g->ops->D + 1) * (size_t)c.n * esz;
    const bool can = c.pattern == PATTERN_PULL2 && c.kernel == KERNEL_NODE && c.bc == LBMK_PERIODIC && !c.Pd.ghost && c.collision == 0;
    const bool cl = can && g->ops->cluster_supported(c);
    if (g->opt_stepping == LBMK_STEPPING_AUTO)
        c.stepping = (cl && g->ops->linear) ? STEPPING_CLUSTER : (can && state2 <= (size_t(96) << 20)) ? STEPPING_PERSISTENT : STEPPING_LAUNCH;
    else if (g->opt_stepping == LBMK_STEPPING_CLUSTER) c.stepping = cl ? STEPPING_CLUSTER : (can ? STEPPING_PERSISTENT : STEPPING_LAUNCH);
    else if (g->opt_stepping == LBMK_STEPPING_RESIDENT) {
        // one population copy in the shared memory of all SMs, AA pattern; grids that do not qualify step as they would have otherwise
        const bool res = c.pattern == PATTERN_AA && c.kernel == KERNEL_NODE && c.bc == LBMK_PERIODIC && !c.Pd.ghost && c.collision == 0 && (c.num_sms <= 0 || g->ops->resident_supported(c));   // SM count known at bind
        c.stepping = res ? STEPPING_RESIDENT : (can && state2 <= (size_t(96) << 20)) ? STEPPING_PERSISTENT : STEPPING_LAUNCH;
    } else c.stepping = (g->opt_stepping == LBMK_STEPPING_PERSISTENT && can) ? STEPPING_PERSISTENT : STEPPING_LAUNCH;
}

static void layout(lbmk_grid* g) {
    GridCore& c = g->c;
    const SysOps* o = g->ops;
    const size_t esz = c.prec == PREC_F64 ? 8 : 4;
    const size_t ntiles = ((size_t)c.n + TILE - 1) / TILE;               // tiled SoA (common.cuh): last tile padded
    const size_t fbytes = align_up((size_t)o->M * (2 * o->D + 1) * ntiles * TILE * esz, 256);
    size_t off = 0;
    g->off_f[0] = off; off += fbytes;
    g->off_f[1] = off; if (c.pattern == PATTERN_PULL2) off += fbytes;
    const int len[3] = {c.nx, c.ny, c.nz};
    for (int a = 0; a < 3; ++a) { g->off_tab[a] = off; off += align_up((size_t)(o->nax[a] > 0 ? o->nax[a] : 1) * len[a] * esz, 256); }
    // per-row forcing coefficients: 2 buffers x coef_B steps x [ny*nz][nc]; a batch is at most ~32 MB and 64 steps
    {
        const size_t per_step = (size_t)(o->nc > 0 ? o->nc : 4) * c.ny * c.nz * esz;
        size_t B = (size_t(32) << 20) / per_step;
        c.coef_B = (int)(B < 1 ? 1 : (B > 64 ? 64 : B));
        if (!(o->has_mms && c.mms_id != 0)) c.coef_B = 1;
        g->off_coef = off; off += align_up(2 * (size_t)c.coef_B * per_step, 256);
    }
    g->off_feq0 = off; off += align_up((size_t)o->M * (2 * o->D + 1) * 8, 256);
    g->off_red = off; off += 256 + (size_t)PERSISTENT_MAX_BLOCKS * FLAG_STRIDE * sizeof(unsigned int);   // [0..3] reductions; then one step flag per block of the persistent kernel
    c.aux_stride = (long long)(ntiles * TILE);
    g->off_aux = off; off += align_up((size_t)(o->n_aux > 0 ? o->n_aux : 0) * ntiles * TILE * esz, 256);
    g->ws_bytes = off;
}

lbmk_status lbmk_grid_create(const lbmk_system* sys, int nx, int ny, int nz, lbmk_bc bc, double dx, double lambda,
                             lbmk_precision precision, void* cuda_stream, lbmk_grid** out) {
    if (!out) return sys_fail(LBMK_EINVAL, "out is NULL");
    *out = nullptr;
    if (!sys) return sys_fail(LBMK_EINVAL, "sys is NULL");
    const SysOps* o = ops_of(sys->id);
    if (nx < 1 || ny < 1 || nz < 1) return sys_fail(LBMK_EINVAL, "grid sizes must be >= 1");
    if (o->D == 2 && nz != 1) return sys_fail(LBMK_EINVAL, "nz must be 1 for a 2D system");
    if ((long long)nx * ny * nz > 0x7fffffffLL) return sys_fail(LBMK_EINVAL, "grid too large: nx*ny*nz must be < 2^31 nodes");
    if (!(dx > 0.0) || !(lambda > 0.0)) return sys_fail(LBMK_EINVAL, "dx and lambda must be > 0");
    if (bc != LBMK_PERIODIC && bc != LBMK_DIRICHLET_MMS) return sys_fail(LBMK_EINVAL, "unknown boundary condition");
    if (precision != LBMK_F64 && precision != LBMK_F32_SHIFTED && precision != LBMK_F64_SHIFTED) return sys_fail(LBMK_EINVAL, "unknown precision");
    if (bc == LBMK_DIRICHLET_MMS && (sys->mms_id == 0 || !o->has_mms))
        return sys_fail(LBMK_EINVAL, "LBMK_DIRICHLET_MMS needs a manufactured solution (lbmk_system_set_mms)");
    if (bc == LBMK_DIRICHLET_MMS && (nx < 3 || ny < 3 || (o->D == 3 && nz < 3))) return sys_fail(LBMK_EINVAL, "bounded grid needs >= 3 nodes per axis");
    // a-priori sub-characteristic check from the declared amplitudes, eq (2.20): s_max/lambda <= c_s
    const double cs = std::sqrt(o->D == 2 ? Lattice<2>::cs2 : Lattice<3>::cs2);
    if (sys->s_max > 0.0 && sys->s_max / lambda > cs) {
        char b[200];
        snprintf(b, sizeof b, "a-priori sub-characteristic violation: s_max/lambda = %.6g > c_s = %.6g", sys->s_max / lambda, cs);
        return sys_fail(LBMK_ESUBCHAR, b);
    }
    lbmk_grid* g = new (std::nothrow) lbmk_grid();
    if (!g) return sys_fail(LBMK_ENOMEM, "host allocation failed");
    g->sys = *sys;
    g->ops = o;
    g->precision = precision;
    g->dx = dx; g->lam = lambda;
    g->opt_pattern = LBMK_PATTERN_AUTO; g->opt_kernel = LBMK_KERNEL_AUTO; g->opt_stepping = LBMK_STEPPING_AUTO;
    g->bound = g->inited = false;
    g->have_events = g->timed = false;
    GridCore& c = g->c;
    memset(&c, 0, sizeof(c));
    c.nx = nx; c.ny = ny; c.nz = nz; c.n = (long long)nx * ny * nz;
    c.prec = precision == LBMK_F32_SHIFTED ? PREC_F32 : PREC_F64;
    c.bc = bc;
    c.mms_id = sys->mms_id;
    c.stream = (cudaStream_t)cuda_stream;
    derive_params(g);
    resolve_options(g);
    layout(g);
    *out = g;
    return LBMK_OK;
}

lbmk_status lbmk_grid_set_option(lbmk_grid* g, lbmk_option key, long long value) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (g->bound) return fail(g, LBMK_ESTATE, "options must be set before the workspace is bound");
    if (key == LBMK_OPT_PATTERN) {
        if (value < LBMK_PATTERN_AUTO || value > LBMK_PATTERN_AA) return fail(g, LBMK_EINVAL, "unknown pattern");
        g->opt_pattern = value;
    } else if (key == LBMK_OPT_KERNEL) {
        if (value < LBMK_KERNEL_AUTO || value > LBMK_KERNEL_TWOPASS) return fail(g, LBMK_EINVAL, "unknown kernel variant");
        if (value == LBMK_KERNEL_ROW) return fail(g, LBMK_EUNSUPPORTED, "LBMK_KERNEL_ROW is reserved: no staged-row kernel in this build");
        g->opt_kernel = value;
    } else if (key == LBMK_OPT_STEPPING) {
        if (value < LBMK_STEPPING_AUTO || value > LBMK_STEPPING_RESIDENT) return fail(g, LBMK_EINVAL, "unknown stepping mode");
        g->opt_stepping = value;
    } else {
        return fail(g, LBMK_EINVAL, "unknown option");
    }
    resolve_options(g);
    layout(g);
    return LBMK_OK;
}

// ------------------------------------------------------------------------------------------------ sub-domains / slabs
static lbmk_status need_inited(lbmk_grid* g);
static lbmk_status need_bound(lbmk_grid* g);
lbmk_status lbmk_grid_set_origin(lbmk_grid* g, int ox, int oy, int oz) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (g->bound) return fail(g, LBMK_ESTATE, "the origin must be set before the workspace is bound");
    GridCore& c = g->c;
    c.Pd.ox = c.Pf.ox = ox; c.Pd.oy = c.Pf.oy = oy; c.Pd.oz = c.Pf.oz = oz;
    return LBMK_OK;
}

lbmk_status lbmk_grid_set_slab(lbmk_grid* g, int enable) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (g->bound) return fail(g, LBMK_ESTATE, "slab mode must be set before the workspace is bound");
    GridCore& c = g->c;
    if (enable) {
        if (c.bc != LBMK_PERIODIC) return fail(g, LBMK_EUNSUPPORTED, "slabs are periodic grids");
        if ((g->ops->D == 3 ? c.nz : c.ny) < 3) return fail(g, LBMK_EINVAL, "a slab needs >= 1 interior plane between its 2 ghost planes");
        g->opt_pattern = LBMK_PATTERN_PULL2;            // the halo is defined on the two-lattice pull storage
        resolve_options(g);
        layout(g);
    }
    c.Pd.ghost = c.Pf.ghost = enable ? 1 : 0;
    resolve_options(g);
    return LBMK_OK;
}

static long long plane_nodes_of(const lbmk_grid* g) { return g->ops->D == 3 ? (long long)g->c.nx * g->c.ny : (long long)g->c.nx; }
static int planes_of(const lbmk_grid* g) { return g->ops->D == 3 ? g->c.nz : g->c.ny; }

lbmk_status lbmk_halo_bytes(const lbmk_grid* g, size_t* bytes) {
    if (!g || !bytes) return sys_fail(LBMK_EINVAL, "NULL argument");
    *bytes = (size_t)g->ops->M * plane_nodes_of(g) * (g->c.prec == PREC_F64 ? 8 : 4);
    return LBMK_OK;
}

static lbmk_status halo_move(lbmk_grid* g, void* lo, void* hi, const bool PACK, void* on_stream) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    GridCore& c = g->c;
    const cudaStream_t hs = on_stream ? (cudaStream_t)on_stream : c.stream;
    if (!c.Pd.ghost) return fail(g, LBMK_ESTATE, "not a slab (lbmk_grid_set_slab)");
    if (!lo || !hi) return fail(g, LBMK_EINVAL, "halo buffer is NULL");
    if (!c.pending) return fail(g, LBMK_ESTATE, "halo exchange is defined after at least one step (initialise the ghost planes through lbmk_init_from_U)");
    const int D = g->ops->D, M = g->ops->M, Q = 2 * D + 1;
    const int up = 2 * D - 1, down = 2 * D;                       // slot of +s / -s along the slowest axis
    const long long pn = plane_nodes_of(g);
    const int np = planes_of(g);
    const unsigned nb = (unsigned)(((long long)M * pn + 255) / 256);
    // pack: lo <- slot(-s) of the first interior plane, hi <- slot(+s) of the last interior plane
    // unpack: lo -> slot(+s) of the lower ghost plane, hi -> slot(-s) of the upper ghost plane
    const int slot_lo = PACK ? down : up, slot_hi = PACK ? up : down;
    const long long plane_lo = PACK ? 1 : 0, plane_hi = PACK ? np - 2 : np - 1;
    void* bufs[2] = {lo, hi};
    const int slots[2] = {slot_lo, slot_hi};
    const long long planes[2] = {plane_lo, plane_hi};
    for (int e = 0; e < 2; ++e) {
        if (c.prec == PREC_F64) {
            if (PACK) halo_kernel<double, true><<<nb, 256, 0, hs>>>((double*)c.f[c.cur], (double*)bufs[e], M, Q, slots[e], planes[e] * pn, pn);
            else halo_kernel<double, false><<<nb, 256, 0, hs>>>((double*)c.f[c.cur], (double*)bufs[e], M, Q, slots[e], planes[e] * pn, pn);
        } else {
            if (PACK) halo_kernel<float, true><<<nb, 256, 0, hs>>>((float*)c.f[c.cur], (float*)bufs[e], M, Q, slots[e], planes[e] * pn, pn);
            else halo_kernel<float, false><<<nb, 256, 0, hs>>>((float*)c.f[c.cur], (float*)bufs[e], M, Q, slots[e], planes[e] * pn, pn);
        }
    }
    c.launches += 2;
    CK(g, cudaGetLastError(), "halo kernel");
    return LBMK_OK;
}
lbmk_status lbmk_halo_pack(lbmk_grid* g, void* send_lo, void* send_hi) { return halo_move(g, send_lo, send_hi, true, nullptr); }
lbmk_status lbmk_halo_unpack(lbmk_grid* g, const void* recv_lo, const void* recv_hi) {
    return halo_move(g, const_cast<void*>(recv_lo), const_cast<void*>(recv_hi), false, nullptr);
}
lbmk_status lbmk_halo_pack_on(lbmk_grid* g, void* send_lo, void* send_hi, void* cuda_stream) { return halo_move(g, send_lo, send_hi, true, cuda_stream); }
lbmk_status lbmk_halo_unpack_on(lbmk_grid* g, const void* recv_lo, const void* recv_hi, void* cuda_stream) {
    return halo_move(g, const_cast<void*>(recv_lo), const_cast<void*>(recv_hi), false, cuda_stream);
}

// One step of a slab, boundary planes first: [first own plane] [last own plane] -> boundary event -> [interior planes].
// The ghost planes are not updated (their face-crossing slots arrive through the halo exchange).
static lbmk_status step_slab_impl(lbmk_grid* g, int peer) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    GridCore& c = g->c;
    if (!c.Pd.ghost) return fail(g, LBMK_ESTATE, "not a slab (lbmk_grid_set_slab)");
    if (peer && !c.peers_set) return fail(g, LBMK_ESTATE, "no halo peers set (lbmk_grid_set_halo_peers)");
    if (peer && (c.collision != 0 || c.kernel != KERNEL_NODE)) return fail(g, LBMK_EUNSUPPORTED, "peer-store halo: BGK with the node kernel only");
    const long long pn = plane_nodes_of(g);
    const int np = planes_of(g);
    long long r[6];
    r[0] = pn; r[1] = 2 * pn;                                           // first own plane
    r[2] = np > 3 ? (long long)(np - 2) * pn : 0; r[3] = np > 3 ? (long long)(np - 1) * pn : 0;   // last own plane (if distinct)
    r[4] = np > 4 ? 2 * pn : 0; r[5] = np > 4 ? (long long)(np - 2) * pn : 0;                      // interior
    CK(g, cudaEventRecord(g->ev0, c.stream), "cudaEventRecord");
    CK(g, g->ops->step_ranges(c, r, g->ev_boundary, peer), "collide_stream launch (slab)");
    CK(g, cudaEventRecord(g->ev1, c.stream), "cudaEventRecord");
    g->timed = true;
    return LBMK_OK;
}
lbmk_status lbmk_step_slab(lbmk_grid* g) { return step_slab_impl(g, 0); }
lbmk_status lbmk_step_slab_peer(lbmk_grid* g) { return step_slab_impl(g, 1); }

lbmk_status lbmk_grid_population_buffers(const lbmk_grid* g, void** f0, void** f1, long long* upper_ghost_first_node) {
    if (!g || !f0 || !f1) return sys_fail(LBMK_EINVAL, "NULL argument");
    if (!g->bound) return sys_fail(LBMK_ESTATE, "no workspace bound");
    *f0 = g->c.f[0]; *f1 = g->c.f[1];
    if (upper_ghost_first_node) *upper_ghost_first_node = (long long)(planes_of(g) - 1) * plane_nodes_of(g);
    return LBMK_OK;
}

lbmk_status lbmk_grid_set_halo_peers(lbmk_grid* g, void* lo_f0, void* lo_f1, long long lo_upper_ghost_first_node, void* hi_f0, void* hi_f1) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    GridCore& c = g->c;
    if (!c.Pd.ghost) return fail(g, LBMK_ESTATE, "not a slab (lbmk_grid_set_slab)");
    if (!lo_f0 || !lo_f1 || !hi_f0 || !hi_f1 || lo_upper_ghost_first_node < 0) return fail(g, LBMK_EINVAL, "bad peer buffers");
    c.peer_f[0][0] = lo_f0; c.peer_f[0][1] = lo_f1; c.peer_f[1][0] = hi_f0; c.peer_f[1][1] = hi_f1;
    c.peer_node0[0] = lo_upper_ghost_first_node;      // lower neighbour: its UPPER ghost plane receives this slab's slot(-s)
    c.peer_node0[1] = 0;                              // upper neighbour: its LOWER ghost plane (plane 0) receives slot(+s)
    c.peers_set = true;
    return LBMK_OK;
}

lbmk_status lbmk_stream_wait_boundary(lbmk_grid* g, void* cuda_stream) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    CK(g, cudaStreamWaitEvent((cudaStream_t)cuda_stream, g->ev_boundary, 0), "cudaStreamWaitEvent");
    return LBMK_OK;
}
lbmk_status lbmk_grid_wait_stream(lbmk_grid* g, void* cuda_stream) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    CK(g, cudaEventRecord(g->ev_join, (cudaStream_t)cuda_stream), "cudaEventRecord");
    CK(g, cudaStreamWaitEvent(g->c.stream, g->ev_join, 0), "cudaStreamWaitEvent");
    return LBMK_OK;
}

lbmk_status lbmk_grid_get_option(const lbmk_grid* g, lbmk_option key, long long* value) {
    if (!g || !value) return sys_fail(LBMK_EINVAL, "NULL argument");
    if (key == LBMK_OPT_PATTERN) *value = g->c.pattern;
    else if (key == LBMK_OPT_KERNEL) *value = g->c.kernel;
    else if (key == LBMK_OPT_STEPPING) *value = g->c.stepping;
    else return sys_fail(LBMK_EINVAL, "unknown option");
    return LBMK_OK;
}

lbmk_status lbmk_grid_workspace_bytes(const lbmk_grid* g, size_t* bytes) {
    if (!g || !bytes) return sys_fail(LBMK_EINVAL, "NULL argument");
    *bytes = g->ws_bytes;
    return LBMK_OK;
}

lbmk_status lbmk_grid_bind_workspace(lbmk_grid* g, void* device_ptr, size_t bytes) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (!device_ptr) return fail(g, LBMK_EINVAL, "workspace pointer is NULL");
    if (((uintptr_t)device_ptr & 255) != 0) return fail(g, LBMK_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < g->ws_bytes) return fail(g, LBMK_ENOMEM, "workspace smaller than lbmk_grid_workspace_bytes");
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, device_ptr);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(g, e, "cudaPointerGetAttributes (no CUDA device? there is no CPU fallback)"); }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return fail(g, LBMK_EINVAL, "workspace is not device memory");
    GridCore& c = g->c;
    char* base = (char*)device_ptr;
    c.f[0] = base + g->off_f[0];
    c.f[1] = c.pattern == PATTERN_PULL2 ? base + g->off_f[1] : nullptr;
    for (int a = 0; a < 3; ++a) c.tab[a] = base + g->off_tab[a];
    c.coef = base + g->off_coef;
    c.feq0 = (double*)(base + g->off_feq0);
    c.red = (unsigned long long*)(base + g->off_red);
    c.bar = (unsigned int*)(base + g->off_red + 256);
    c.aux_buf = g->ops->n_aux > 0 ? base + g->off_aux : nullptr;
    c.aux_set = false;
    c.cur = 0;
    {
        int dev = 0, sms = 0;
        CK(g, cudaGetDevice(&dev), "cudaGetDevice");
        CK(g, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
        c.num_sms = sms;
        if (c.stepping == STEPPING_RESIDENT && !g->ops->resident_supported(c)) c.stepping = STEPPING_LAUNCH;   // does not fit this GPU's shared memory
    }
    CK(g, g->ops->fill_tables(c), "fill_tables");
    CK(g, g->ops->reference_equilibrium(c), "reference_equilibrium");
    if (!g->have_events) {
        CK(g, cudaEventCreate(&g->ev0), "cudaEventCreate");
        CK(g, cudaEventCreate(&g->ev1), "cudaEventCreate");
        CK(g, cudaStreamCreateWithFlags(&c.aux, cudaStreamNonBlocking), "cudaStreamCreate");
        CK(g, cudaEventCreateWithFlags(&c.ev_entry, cudaEventDisableTiming), "cudaEventCreate");
        CK(g, cudaEventCreateWithFlags(&g->ev_boundary, cudaEventDisableTiming), "cudaEventCreate");
        CK(g, cudaEventCreateWithFlags(&g->ev_join, cudaEventDisableTiming), "cudaEventCreate");
        for (int b = 0; b < 2; ++b) {
            CK(g, cudaEventCreateWithFlags(&c.ev_coef[b], cudaEventDisableTiming), "cudaEventCreate");
            CK(g, cudaEventCreateWithFlags(&c.ev_free[b], cudaEventDisableTiming), "cudaEventCreate");
        }
        g->have_events = true;
    }
    g->bound = true;
    g->inited = false;
    return LBMK_OK;
}

void lbmk_grid_destroy(lbmk_grid* g) {
    if (!g) return;
    if (g->have_events) {
        cudaStreamSynchronize(g->c.aux);
        cudaEventDestroy(g->ev0); cudaEventDestroy(g->ev1); cudaEventDestroy(g->c.ev_entry);
        cudaEventDestroy(g->ev_boundary); cudaEventDestroy(g->ev_join);
        for (int b = 0; b < 2; ++b) { cudaEventDestroy(g->c.ev_coef[b]); cudaEventDestroy(g->c.ev_free[b]); }
        cudaStreamDestroy(g->c.aux);
    }
    delete g;
}

// ------------------------------------------------------------------------------------------------ data in/out
// Stage `bytes` of host data into a transient stream-ordered device buffer (or pass a device pointer through).
struct Staging {
    void* dev = nullptr;
    bool owned = false;
    cudaStream_t stream = nullptr;
    cudaError_t acquire(const void* user, int on_device, size_t bytes, bool copy_in, cudaStream_t s) {
        stream = s;
        if (on_device) { dev = const_cast<void*>(user); return cudaSuccess; }
        cudaError_t e = cudaMallocAsync(&dev, bytes, s);
        if (e != cudaSuccess) return e;
        owned = true;
        if (copy_in) e = cudaMemcpyAsync(dev, user, bytes, cudaMemcpyHostToDevice, s);
        return e;
    }
    cudaError_t release() {
        if (!owned) return cudaSuccess;
        owned = false;
        return cudaFreeAsync(dev, stream);
    }
    ~Staging() { if (owned) cudaFreeAsync(dev, stream); }
};

static lbmk_status need_bound(lbmk_grid* g) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (!g->bound) return fail(g, LBMK_ESTATE, "no workspace bound (lbmk_grid_bind_workspace)");
    return LBMK_OK;
}
static lbmk_status need_inited(lbmk_grid* g) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    if (!g->inited) return fail(g, LBMK_ESTATE, "grid not initialised (lbmk_init_from_U)");
    return LBMK_OK;
}

// Host <-> device transfer of U [m_total][n] in NODE CHUNKS through two fixed staging buffers (2 x ~32 MB) on the auxiliary stream:
// the copy of chunk j+1 overlaps the kernel on chunk j, and no second device copy of U is ever allocated (the 256^3 17-field
// headline grid has a 2.3 GB fp64 U).  Each chunk is a strided 2D copy: m_total rows of `w` nodes, n apart on the host.
static long long chunk_nodes(int M, long long n) {
    long long c = (long long)((size_t(32) << 20) / ((size_t)M * sizeof(double))) / TILE * TILE;
    if (c < TILE) c = TILE;
    return c < n ? c : n;
}

static lbmk_status host_init_chunked(lbmk_grid* g, const double* U) {
    GridCore& c = g->c;
    const int M = g->ops->M;
    const long long C = chunk_nodes(M, c.n);
    double* stage = nullptr;
    CK(g, cudaMallocAsync((void**)&stage, 2 * (size_t)M * C * sizeof(double), c.stream), "cudaMallocAsync staging");
    cudaError_t e = cudaEventRecord(c.ev_entry, c.stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c.aux, c.ev_entry, 0);
    long long j = 0;
    for (long long node0 = 0; node0 < c.n && e == cudaSuccess; node0 += C, ++j) {
        const int b = (int)(j & 1);
        const long long node1 = node0 + C < c.n ? node0 + C : c.n, w = node1 - node0;
        double* sb = stage + (size_t)b * M * C;
        if (j >= 2) e = cudaStreamWaitEvent(c.aux, c.ev_free[b], 0);               // the kernel on chunk j-2 has consumed this buffer
        if (e == cudaSuccess) e = cudaMemcpy2DAsync(sb, (size_t)C * sizeof(double), U + node0, (size_t)c.n * sizeof(double), (size_t)w * sizeof(double),
                                                    (size_t)M, cudaMemcpyHostToDevice, c.aux);
        if (e == cudaSuccess) e = cudaEventRecord(c.ev_coef[b], c.aux);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c.stream, c.ev_coef[b], 0);
        if (e == cudaSuccess) e = g->ops->init_range(c, sb, C, node0, node1);
        if (e == cudaSuccess) e = cudaEventRecord(c.ev_free[b], c.stream);
    }
    cudaError_t e2 = cudaFreeAsync(stage, c.stream);
    cudaError_t e3 = cudaStreamSynchronize(c.stream);                               // the host buffer is only borrowed
    CK(g, e, "chunked init_from_U");
    CK(g, e2, "cudaFreeAsync");
    CK(g, e3, "cudaStreamSynchronize");
    return LBMK_OK;
}

static lbmk_status host_read_chunked(lbmk_grid* g, double* U_out) {
    GridCore& c = g->c;
    const int M = g->ops->M;
    const long long C = chunk_nodes(M, c.n);
    CK(g, g->ops->frame_now(c), "frame refresh");
    double* stage = nullptr;
    CK(g, cudaMallocAsync((void**)&stage, 2 * (size_t)M * C * sizeof(double), c.stream), "cudaMallocAsync staging");
    cudaError_t e = cudaSuccess;
    long long j = 0;
    for (long long node0 = 0; node0 < c.n && e == cudaSuccess; node0 += C, ++j) {
        const int b = (int)(j & 1);
        const long long node1 = node0 + C < c.n ? node0 + C : c.n, w = node1 - node0;
        double* sb = stage + (size_t)b * M * C;
        if (j >= 2) e = cudaStreamWaitEvent(c.stream, c.ev_free[b], 0);            // the copy of chunk j-2 has left this buffer
        if (e == cudaSuccess) e = g->ops->read_range(c, sb, C, node0, node1);
        if (e == cudaSuccess) e = cudaEventRecord(c.ev_coef[b], c.stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c.aux, c.ev_coef[b], 0);
        if (e == cudaSuccess) e = cudaMemcpy2DAsync(U_out + node0, (size_t)c.n * sizeof(double), sb, (size_t)C * sizeof(double), (size_t)w * sizeof(double),
                                                    (size_t)M, cudaMemcpyDeviceToHost, c.aux);
        if (e == cudaSuccess) e = cudaEventRecord(c.ev_free[b], c.aux);
    }
    for (int b = 0; b < 2 && b < j; ++b) { cudaError_t ew = cudaStreamWaitEvent(c.stream, c.ev_free[b], 0); if (e == cudaSuccess) e = ew; }
    cudaError_t e2 = cudaFreeAsync(stage, c.stream);
    cudaError_t e3 = cudaStreamSynchronize(c.stream);
    CK(g, e, "chunked read_U");
    CK(g, e2, "cudaFreeAsync");
    CK(g, e3, "cudaStreamSynchronize");
    return LBMK_OK;
}

lbmk_status lbmk_init_from_U(lbmk_grid* g, const double* U, int on_device, double t0) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    if (!U) return fail(g, LBMK_EINVAL, "U is NULL");
    GridCore& c = g->c;
    if (g->ops->n_aux > 0 && !c.aux_set) return fail(g, LBMK_ESTATE, "this system has prescribed coefficient fields: call lbmk_set_aux_fields first");
    c.step = 0; c.t0 = t0; c.cur = 0;
    if (on_device) CK(g, g->ops->init_from_U(c, U), "init_from_U kernel");
    else {
        s = host_init_chunked(g, U);
        if (s != LBMK_OK) return s;
    }
    g->inited = true;
    return LBMK_OK;
}

lbmk_status lbmk_set_aux_fields(lbmk_grid* g, const double* A, int on_device) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    if (!A) return fail(g, LBMK_EINVAL, "A is NULL");
    if (g->ops->n_aux == 0) return fail(g, LBMK_EUNSUPPORTED, "this system has no prescribed coefficient fields");
    GridCore& c = g->c;
    const size_t bytes = (size_t)g->ops->n_aux * c.n * sizeof(double);
    Staging st;
    CK(g, st.acquire(A, on_device, bytes, true, c.stream), "stage A");
    CK(g, g->ops->set_aux(c, (const double*)st.dev), "set_aux kernel");
    CK(g, st.release(), "cudaFreeAsync");
    if (!on_device) CK(g, cudaStreamSynchronize(c.stream), "cudaStreamSynchronize");
    return LBMK_OK;
}

lbmk_status lbmk_set_populations(lbmk_grid* g, const double* f, int on_device, double t0) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    if (!f) return fail(g, LBMK_EINVAL, "f is NULL");
    GridCore& c = g->c;
    if (g->ops->n_aux > 0 && !c.aux_set) return fail(g, LBMK_ESTATE, "this system has prescribed coefficient fields: call lbmk_set_aux_fields first");
    const size_t bytes = (size_t)g->ops->M * (2 * g->ops->D + 1) * c.n * sizeof(double);
    Staging st;
    CK(g, st.acquire(f, on_device, bytes, true, c.stream), "stage f");
    c.step = 0; c.t0 = t0; c.cur = 0;
    CK(g, g->ops->set_f(c, (const double*)st.dev), "set_f kernel");
    CK(g, st.release(), "cudaFreeAsync");
    if (!on_device) CK(g, cudaStreamSynchronize(c.stream), "cudaStreamSynchronize");
    g->inited = true;
    return LBMK_OK;
}

lbmk_status lbmk_step(lbmk_grid* g, int n_steps) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    if (n_steps < 0) return fail(g, LBMK_EINVAL, "n_steps must be >= 0");
    if (n_steps == 0) return LBMK_OK;
    GridCore& c = g->c;
    CK(g, cudaEventRecord(g->ev0, c.stream), "cudaEventRecord");
    CK(g, g->ops->step(c, n_steps), "collide_stream launch");
    CK(g, cudaEventRecord(g->ev1, c.stream), "cudaEventRecord");
    g->timed = true;
    return LBMK_OK;
}

lbmk_status lbmk_last_step_ms(lbmk_grid* g, float* ms) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    if (!ms) return fail(g, LBMK_EINVAL, "ms is NULL");
    if (!g->timed) return fail(g, LBMK_ESTATE, "no lbmk_step call to time yet");
    CK(g, cudaEventSynchronize(g->ev1), "cudaEventSynchronize");
    CK(g, cudaEventElapsedTime(ms, g->ev0, g->ev1), "cudaEventElapsedTime");
    return LBMK_OK;
}

lbmk_status lbmk_read_U(lbmk_grid* g, double* U_out, int on_device) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    if (!U_out) return fail(g, LBMK_EINVAL, "U_out is NULL");
    GridCore& c = g->c;
    if (!on_device) return host_read_chunked(g, U_out);
    CK(g, g->ops->read_U(c, U_out), "read_U kernel");
    CK(g, cudaStreamSynchronize(c.stream), "cudaStreamSynchronize");
    return LBMK_OK;
}

lbmk_status lbmk_read_populations(lbmk_grid* g, double* f_out, int on_device) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    if (!f_out) return fail(g, LBMK_EINVAL, "f_out is NULL");
    GridCore& c = g->c;
    const size_t bytes = (size_t)g->ops->M * (2 * g->ops->D + 1) * c.n * sizeof(double);
    Staging st;
    CK(g, st.acquire(f_out, on_device, bytes, false, c.stream), "stage f_out");
    CK(g, g->ops->read_f(c, (double*)st.dev), "read_f kernel");
    if (!on_device) CK(g, cudaMemcpyAsync(f_out, st.dev, bytes, cudaMemcpyDeviceToHost, c.stream), "cudaMemcpyAsync D2H");
    CK(g, st.release(), "cudaFreeAsync");
    CK(g, cudaStreamSynchronize(c.stream), "cudaStreamSynchronize");
    return LBMK_OK;
}

lbmk_status lbmk_time(const lbmk_grid* g, long long* step, double* t) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (step) *step = g->c.step;
    if (t) *t = g->c.t0 + (double)g->c.step * g->c.dt;
    return LBMK_OK;
}

lbmk_status lbmk_check_subcharacteristic(lbmk_grid* g, double* out3) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    double o[3];
    CK(g, g->ops->max_wave_speed(g->c, o), "max_wave_speed kernel");
    if (out3) { out3[0] = o[0]; out3[1] = o[1]; out3[2] = o[2]; }
    const double cs = std::sqrt(g->ops->D == 2 ? Lattice<2>::cs2 : Lattice<3>::cs2);
    const double sp = std::fmax(o[0], o[1]) + o[2];
    if (!(sp <= cs)) {
        char b[200];
        snprintf(b, sizeof b, "sub-characteristic violation: lattice wave speed %.6g > c_s = %.6g", sp, cs);
        return fail(g, LBMK_ESUBCHAR, b);
    }
    return LBMK_OK;
}

lbmk_status lbmk_error_norms(lbmk_grid* g, double* out) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    if (!out) return fail(g, LBMK_EINVAL, "out is NULL");
    GridCore& c = g->c;
    if (!g->ops->has_mms || c.mms_id == 0) return fail(g, LBMK_EUNSUPPORTED, "error norms need a manufactured solution (lbmk_system_set_mms)");
    const size_t bytes = (size_t)g->ops->M * 6 * sizeof(double);
    Staging st;
    CK(g, st.acquire(out, 0, bytes, false, c.stream), "stage norms");
    CK(g, g->ops->error_norms(c, (double*)st.dev), "error_norms kernel");
    CK(g, cudaMemcpyAsync(out, st.dev, bytes, cudaMemcpyDeviceToHost, c.stream), "cudaMemcpyAsync D2H");
    CK(g, cudaStreamSynchronize(c.stream), "cudaStreamSynchronize");
    CK(g, st.release(), "cudaFreeAsync");
    return LBMK_OK;
}

// ---- error norms without any allocation (lbmk.h lbmk_error_norms_noalloc)
// The scratch of the two-pass reduction lives in this file-scope device array: LBMK_NOALLOC_SCRATCH_BYTES on every GPU that loads
// the library, until exit.  In host code `noalloc_scratch` is only the host-side stand-in of the symbol, NOT a device address: the
// device address is looked up once per device with cudaGetSymbolAddress, with that device current, and that pointer is what the
// kernels get.  All calls on a device share the array (it keeps the last call's contents; pass 1 overwrites every record it will
// read, so nothing has to be cleared), hence calls that overlap on the GPU race.
static __device__ __align__(256) unsigned char noalloc_scratch[LBMK_NOALLOC_SCRATCH_BYTES];

static constexpr int NOALLOC_MAX_DEVICES = 64;
static std::mutex noalloc_mutex;
static void* noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

static cudaError_t noalloc_scratch_address(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(noalloc_mutex);
    if (!noalloc_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, noalloc_scratch);       // the current device's instance of the array
        if (e != cudaSuccess) return e;
        noalloc_ptr[dev] = p;
    }
    *out = noalloc_ptr[dev];
    return cudaSuccess;
}

lbmk_status lbmk_error_norms_noalloc(lbmk_grid* g, double* out_device) {
    if (!g) return sys_fail(LBMK_EINVAL, "grid is NULL");
    if (!out_device) return fail(g, LBMK_EINVAL, "out_device is NULL");
    GridCore& c = g->c;
    if (!g->ops->has_mms || c.mms_id == 0) return fail(g, LBMK_EUNSUPPORTED, "error norms need a manufactured solution (lbmk_system_set_mms)");
    // size first: it is a property of the grid, known before any workspace is bound
    const long long nrec = (c.n + NORM_RECORD_NODES - 1) / NORM_RECORD_NODES;
    const size_t need = (size_t)nrec * g->ops->M * 6 * sizeof(double);
    if (need > (size_t)LBMK_NOALLOC_SCRATCH_BYTES) {
        char msg[256];
        snprintf(msg, sizeof msg, "grid too large for the static scratch of lbmk_error_norms_noalloc: %lld records of %d x 6 doubles = %zu bytes, "
                 "the array holds %d bytes (use lbmk_error_norms)", nrec, g->ops->M, need, (int)LBMK_NOALLOC_SCRATCH_BYTES);
        return fail(g, LBMK_EINVAL, msg);
    }
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    void* scratch = nullptr;
    CK(g, noalloc_scratch_address(&scratch), "cudaGetSymbolAddress(noalloc_scratch)");
    CK(g, g->ops->error_norm_records(c, (double*)scratch, out_device), "error_norm_records kernels");
    return LBMK_OK;                                          // asynchronous on the grid's stream, like lbmk_step
}

// ---- generated augmented systems (gen/cascade.py -> cascade_generated.cuh)
lbmk_status lbmk_generated_flux(lbmk_system_id id, const double* U, const double* A, const double* params, int n_params,
                                double dx, double lambda, double g_tau, double* F_out, double* S_out) {
    if (!U || !F_out || !S_out) return sys_fail(LBMK_EINVAL, "NULL argument");
    if (id < 0 || id >= LBMK_SYS_COUNT || n_params != N_PARAMS[id] || (n_params > 0 && !params)) return sys_fail(LBMK_EINVAL, "unknown system or wrong parameter count");
    if (!(dx > 0.0) || !(lambda > 0.0) || !(g_tau > 0.0)) return sys_fail(LBMK_EINVAL, "dx, lambda, g_tau must be > 0");
    GenArgs<double> ga;
    memset(&ga, 0, sizeof ga);
    for (int i = 0; i < n_params; ++i) ga.par[i] = params[i];
    ga.dx = dx; ga.dt = dx / lambda; ga.gtau = g_tau;
    switch (id) {
        case LBMK_SYS_EULER2D: gen_eval<Gen_euler2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_SWE2D_BATHY: gen_eval<Gen_swe2d_bathy>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_ADR2D: gen_eval<Gen_adr2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_ALLENCAHN2D: gen_eval<Gen_allencahn2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_INSE2D: gen_eval<Gen_inse2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_NSF2D_GRADTRACK: gen_eval<Gen_nsf2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_MHD2D: gen_eval<Gen_mhd2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_NSF3D_GRADTRACK: gen_eval<Gen_nsf3d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_ADVECTION2D: gen_eval<Gen_advection2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_BURGERS2D: gen_eval<Gen_burgers2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_SWE2D: gen_eval<Gen_swe2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_URF2D: gen_eval<Gen_urf2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_MAXWELL2D: gen_eval<Gen_maxwell2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_ELASTICITY2D: gen_eval<Gen_elasticity2d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_HCNSF3D: gen_eval<Gen_hcnsf3d>(U, A, ga, F_out, S_out); break;
        case LBMK_SYS_MHD3D_JTRACK: gen_eval<Gen_mhd3d>(U, A, ga, F_out, S_out); break;
        default: return sys_fail(LBMK_EUNSUPPORTED, "no generated augmented system for this id (gen/cascade.py)");
    }
    return LBMK_OK;
}

lbmk_status lbmk_flux_selfcheck(lbmk_grid* g, double* max_rel_diff) {
    lbmk_status s = need_inited(g);
    if (s != LBMK_OK) return s;
    if (!max_rel_diff) return fail(g, LBMK_EINVAL, "output is NULL");
    if (!g->ops->has_generated) return fail(g, LBMK_EUNSUPPORTED, "no generated augmented system for this system (gen/cascade.py)");
    CK(g, g->ops->flux_selfcheck(g->c, g->sys.g_tau, max_rel_diff), "flux_selfcheck kernel");
    return LBMK_OK;
}

lbmk_status lbmk_stream_index_map(lbmk_grid* g, int dir, long long* src_index_out, int on_device) {
    lbmk_status s = need_bound(g);
    if (s != LBMK_OK) return s;
    if (!src_index_out) return fail(g, LBMK_EINVAL, "output is NULL");
    if (dir < 0 || dir > 2 * g->ops->D) return fail(g, LBMK_EINVAL, "direction out of range");
    GridCore& c = g->c;
    const size_t bytes = (size_t)c.n * sizeof(long long);
    Staging st;
    CK(g, st.acquire(src_index_out, on_device, bytes, false, c.stream), "stage index map");
    stream_index_map_kernel<<<(unsigned)((c.n + 255) / 256), 256, 0, c.stream>>>((long long*)st.dev, dir, c.nx, c.ny, c.nz, c.n);
    c.launches++;
    CK(g, cudaGetLastError(), "stream_index_map kernel");
    if (!on_device) CK(g, cudaMemcpyAsync(src_index_out, st.dev, bytes, cudaMemcpyDeviceToHost, c.stream), "cudaMemcpyAsync D2H");
    CK(g, st.release(), "cudaFreeAsync");
    CK(g, cudaStreamSynchronize(c.stream), "cudaStreamSynchronize");
    return LBMK_OK;
}

lbmk_status lbmk_grid_omega(const lbmk_grid* g, double* omega_out) {
    if (!g || !omega_out) return sys_fail(LBMK_EINVAL, "NULL argument");
    for (int k = 0; k < g->ops->M; ++k) omega_out[k] = g->c.Pd.omega[k];
    return LBMK_OK;
}

lbmk_status lbmk_grid_omega_plus(const lbmk_grid* g, double* omega_out) {
    if (!g || !omega_out) return sys_fail(LBMK_EINVAL, "NULL argument");
    for (int k = 0; k < g->ops->M; ++k) omega_out[k] = g->c.Pd.omega_p[k];
    return LBMK_OK;
}

lbmk_status lbmk_grid_launch_count(const lbmk_grid* g, long long* launches) {
    if (!g || !launches) return sys_fail(LBMK_EINVAL, "NULL argument");
    *launches = g->c.launches;
    return LBMK_OK;
}

lbmk_status lbmk_copy_bandwidth(void* dst, const void* src, size_t bytes, int reps, void* cuda_stream, double* gbs) {
    if (!dst || !src || !gbs || reps < 1 || bytes < 16) return sys_fail(LBMK_EINVAL, "bad argument");
    if ((((uintptr_t)dst) | ((uintptr_t)src)) & 15) return sys_fail(LBMK_EINVAL, "pointers must be 16-byte aligned");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaEvent_t a, b;
    cudaError_t e;
    if ((e = cudaEventCreate(&a)) != cudaSuccess) return cuda_fail(nullptr, e, "cudaEventCreate");
    if ((e = cudaEventCreate(&b)) != cudaSuccess) { cudaEventDestroy(a); return cuda_fail(nullptr, e, "cudaEventCreate"); }
    const size_t n16 = bytes / 16;
    const unsigned nb = (unsigned)((n16 + 1023) / 1024);
    copy_kernel<<<nb, 256, 0, s>>>((float4*)dst, (const float4*)src, n16);   // warm-up
    cudaEventRecord(a, s);
    for (int r = 0; r < reps; ++r) copy_kernel<<<nb, 256, 0, s>>>((float4*)dst, (const float4*)src, n16);
    cudaEventRecord(b, s);
    e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "copy_kernel");
    *gbs = 2.0 * (double)(n16 * 16) * reps / (ms * 1e-3) / 1e9;
    return LBMK_OK;
}

}  // extern "C"
