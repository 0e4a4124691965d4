/* lbmk.h -- C-ABI of the B200-native collide-and-stream library (liblbmk.so).
 *
 * One thing is implemented behind this boundary: the fused collide-and-stream time step of the
 * vector-population discrete-kinetic relaxation LBM of arxiv/paper_2607_05668 for a system of m
 * conservation laws  d_t Q + div Phi(Q) = S  (eq 2.1):
 *   - every component k of the augmented state Q+ (conserved fields + the gradient-tracker fields the
 *     first-order cascade adds, eq 2.2-2.4) carries its own Q populations f_k,i on
 *     one compact lattice, D2Q5 or D3Q7 (eq 2.5-2.6; Table SM1);
 *   - exact-flux equilibrium  f_eq,k,i = w_i (Q_k + c_i . F_k / c_s^2),  F_k = (dt/dx) Phi_k(Q+)
 *     (eq 2.7-2.8);
 *   - BGK collide-and-stream with the source taken as w_i dt S (eq 2.11);
 *   - fp64, or the reference- and equilibrium-shifted fp32 form f* = f - f_eq(Q0, F0)
 *     (eq 2.23).
 * The call sequence follows the paper's statement of the problem: declare the system (m, lattice,
 * flux/source specialisation, relaxation times, lattice velocity), allocate a periodic or bounded grid,
 * initialise from U, step N times, read back U.
 *
 * Conventions
 *   - Every function returns lbmk_status; no exception crosses the ABI.  On failure the grid (or, for
 *     system calls, a thread-local slot) keeps a message readable with lbmk_last_error().
 *   - Handles (lbmk_system*, lbmk_grid*) are library-owned and freed by the *_destroy calls.
 *   - Population memory is CALLER-owned device memory (e.g. a torch tensor): query the size with
 *     lbmk_grid_workspace_bytes(), allocate, hand it over with lbmk_grid_bind_workspace().  The library
 *     never frees it.  Arrays passed to init/read calls are borrowed for the duration of the call.
 *   - "on_device" arguments say whether a data pointer is a DEVICE pointer (non-zero) or a HOST pointer
 *     (zero).  Host U arrays (lbmk_init_from_U, lbmk_read_U) move in node chunks through two fixed ~32 MB stream-ordered staging
 *     buffers, the copy of one chunk overlapping the kernel on the other (pinned host memory makes the copies asynchronous);
 *     the other host transfers are staged through a transient stream-ordered device allocation of their own size.
 *   - All work is enqueued on the cudaStream_t given to lbmk_grid_create (passed as void*; NULL = the
 *     legacy default stream).  lbmk_step is asynchronous; calls that return data to the host synchronise
 *     that stream.
 *   - Field layout everywhere: U[k][z][y][x] and f[k][i][z][y][x], C-contiguous, x fastest, nz = 1 in 2D.
 *     Node coordinates x_j = j*dx.  Direction order i: 0 rest; 1:+x 2:-x 3:+y 4:-y 5:+z 6:-z.
 *   - There is NO CPU fallback: without a CUDA device every compute call returns LBMK_ECUDA.
 */
#ifndef LBMK_H
#define LBMK_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LBMK_MAX_COMPONENTS 32
#define LBMK_MAX_PARAMS 16

typedef enum {
    LBMK_OK = 0,
    LBMK_EINVAL = 1,       /* bad argument: unknown id, non-positive size, NULL pointer, wrong count */
    LBMK_ENOMEM = 2,       /* workspace too small / host allocation failed */
    LBMK_ECUDA = 3,        /* a CUDA runtime call failed (message holds cudaGetErrorString) */
    LBMK_ESUBCHAR = 4,     /* sub-characteristic condition violated (eq 2.19-2.20) */
    LBMK_ESTATE = 5,       /* call out of order (e.g. step before init, bind after init) */
    LBMK_EUNSUPPORTED = 6  /* valid request this build has no kernel for */
} lbmk_status;

typedef enum { LBMK_D2Q5 = 0, LBMK_D3Q7 = 1 } lbmk_lattice;          /* Table SM1 */
typedef enum { LBMK_F64 = 0, LBMK_F32_SHIFTED = 1,                   /* eq 2.23 */
               LBMK_F64_SHIFTED = 2 /* shift algebra in fp64: test of the identity */ } lbmk_precision;
typedef enum { LBMK_PERIODIC = 0, LBMK_DIRICHLET_MMS = 1 } lbmk_bc;

/* Compiled-in flux/source specialisations (the paper's Emit stage, Alg 2.1 lines 24-25, replaced by
 * hand-written / build-time generated CUDA).  params order per system:
 *   ADVECTION2D  {a_x, a_y}            Phi = a U                                   m = 1
 *   BURGERS2D    {}                    Phi = (u^2/2, u^2/2)   eq 3.1-3.2 L317-L323 m = 1
 *   SWE2D        {g}                   eq 3.6, flat bottom               m = 3 (h, hu, hv)
 *   EULER2D      {gamma}               eq 3.4 L344-L347                            m = 4 (rho, mx, my, E)
 *   ADR2D        {u_x, u_y, D, R}      eq 3.17 L424-L425                           m = 1 + 2 trackers
 *   NSF3D        {gamma, mu, K}        eq 3.23 L456-L463 + trackers of grad u (9), grad T (3)  m = 5 + 12
 *   MHD3D        {gamma, eta}          eq 3.25, current-density trackers J (3)       m = 8 + 3
 *   URF2D        {}                    ideal ultrarelativistic fluid, eq 3.7-3.9 L365-L381     m = 3 (E, S_x, S_y)
 *   ALLENCAHN2D  {gamma, r}            Allen-Cahn phase field, eq 3.18-3.19 L429-L434          m = 1 + 2 trackers
 *   INSE2D       {c_s_phys, mu}        weakly compressible NSE, eq 3.21-3.22 L446-L452          m = 3 + 4 trackers
 *   ELASTICITY2D {rho0, mu_s, lambda_s} neo-Hookean finite-strain elasticity, eq 3.13-3.15 L402-L414  m = 6 (F, rho0 v)
 *   NSF2D        {gamma, mu, K}        compressible NSF 2D, eq 3.23-3.24, cascade on the conserved fields  m = 4 + 8
 *   MAXWELL2D    {c}                   Maxwell TM mode, eq 3.10-3.11 L385-L391                 m = 3 (E_z, H_x, H_y)
 *   SWE2D_BATHY  {g}                   eq 3.5-3.6 L351-L359 with the bed source -g h grad z_b  m = 3; 2 prescribed fields (d_x z_b, d_y z_b)
 *   HCNSF3D      {gamma, mu, kappa, eta_drag}  homogenized NSF, eq 3.27, trackers sym grad u (6: 00 11 22 01 02 12),
 *                                      grad T (3)                                              m = 5 + 9; 4 prescribed fields (alpha, u_s x3)
 *   MHD2D        {gamma, mu, K, eta}   resistive MHD 2D with Powell source, eq 3.25, cascade on the 6 conserved
 *                                      fields (rho, m0, m1, E, B0, B1)                          m = 6 + 12
 * Trackers are carried in lattice units G^L = dx grad V.
 * Prescribed coefficient fields ("prescribed external coefficient fields [that] enter the dynamics without being functions
 * of the evolved state") are per-node inputs set with lbmk_set_aux_fields. */
typedef enum {
    LBMK_SYS_ADVECTION2D = 0, LBMK_SYS_BURGERS2D = 1, LBMK_SYS_SWE2D = 2, LBMK_SYS_EULER2D = 3,
    LBMK_SYS_ADR2D = 4, LBMK_SYS_NSF3D_GRADTRACK = 5, LBMK_SYS_MHD3D_JTRACK = 6, LBMK_SYS_URF2D = 7,
    LBMK_SYS_MAXWELL2D = 8, LBMK_SYS_ALLENCAHN2D = 9, LBMK_SYS_INSE2D = 10,
    LBMK_SYS_ELASTICITY2D = 11, LBMK_SYS_NSF2D_GRADTRACK = 12, LBMK_SYS_SWE2D_BATHY = 13, LBMK_SYS_HCNSF3D = 14,
    LBMK_SYS_MHD2D = 15, LBMK_SYS_COUNT = 16
} lbmk_system_id;

/* Grid options (lbmk_grid_set_option, before lbmk_grid_workspace_bytes / bind). */
typedef enum {
    LBMK_OPT_PATTERN = 0,   /* streaming pattern: LBMK_PATTERN_* ; default chosen per config by measurement */
    LBMK_OPT_KERNEL = 1,    /* kernel variant: LBMK_KERNEL_* */
    LBMK_OPT_STEPPING = 2   /* how lbmk_step(n) issues its n steps: LBMK_STEPPING_* */
} lbmk_option;
/* LBMK_STEPPING_LAUNCH: one kernel launch per step.  LBMK_STEPPING_PERSISTENT: one cooperative launch advances a whole batch
 * of steps (all blocks co-resident, point-to-point step flags between neighbouring blocks) -- for grids whose populations live in L2 and whose
 * step is therefore launch-latency bound (SURVEY.md section 7 "Small configs"); two-lattice pull, periodic, node kernel only,
 * bit-identical to the per-launch path.  LBMK_STEPPING_CLUSTER: grids of at most 8192 nodes of a small tracker-free system
 * without forcing or prescribed fields (configs[0]): ONE thread-block cluster of 8 CTAs keeps the populations in distributed
 * shared memory for the whole lbmk_step(n) call, one hardware cluster barrier per step; same arithmetic, equal to the other
 * paths to rounding (nvcc decides FMA contraction per kernel; bit-identical for linear systems such as configs[0]'s).
 * AUTO never changes bits: it picks CLUSTER only when the grid qualifies AND the system is linear (configs[0]), else PERSISTENT
 * when both population copies fit in 96 MB, else LAUNCH; CLUSTER for a nonlinear system must be asked for explicitly; a mode
 * the grid does not qualify for falls back to the next one (lbmk_grid_get_option returns the resolved mode).
 * LBMK_STEPPING_RESIDENT (never picked by AUTO): grids whose ONE population copy fits in the shared memory of all SMs together
 * (148 x 227 KB = 33 MB; configs[1] in fp64 is 31 MB): one cooperative launch with one block per SM, every block keeps its
 * contiguous run of 128-node tiles in shared memory and steps it in place with the AA pattern; only the populations that cross a
 * block boundary stay in global memory (L2).  Implies LBMK_PATTERN_AA unless a pattern was set; periodic, node kernel, BGK;
 * any system, forcing and prescribed fields included.  Same arithmetic (collide_core), equal to the other paths to rounding.
 * Resolved at lbmk_grid_bind_workspace (the SM count is a property of the device): a grid that does not fit steps per launch. */
enum { LBMK_STEPPING_AUTO = 0, LBMK_STEPPING_LAUNCH = 1, LBMK_STEPPING_PERSISTENT = 2, LBMK_STEPPING_CLUSTER = 3, LBMK_STEPPING_RESIDENT = 4 };
enum { LBMK_PATTERN_AUTO = 0, LBMK_PATTERN_PULL2 = 1 /* two-lattice pull */, LBMK_PATTERN_AA = 2 /* in-place */ };
enum { LBMK_KERNEL_AUTO = 0, LBMK_KERNEL_NODE = 1 /* one node per thread, direct loads */,
       LBMK_KERNEL_ROW = 2 /* reserved: shared-memory / TMA staged x-rows; not built (direct loads already move exactly the
                              algorithmic bytes at the copy peak) -- selecting it returns LBMK_EUNSUPPORTED */,
       LBMK_KERNEL_TWOPASS = 3 /* one node per thread, moments first, populations re-read for the relaxation */ };

typedef struct lbmk_system lbmk_system;
typedef struct lbmk_grid lbmk_grid;

/* ---- declare the system (eq 2.1; Alg 2.1 "Split/Cascade/Assemble" results are compiled in) ---------- */

/* Creates a system.  lattice must match the system's dimension (2D: D2Q5, 3D: D3Q7).  params: n_params
 * doubles in the order listed above (host pointer, copied).  *out receives the handle. */
lbmk_status lbmk_system_create(lbmk_system_id id, lbmk_lattice lattice, const double* params, int n_params,
                               lbmk_system** out);
/* m_conserved, m_total (= conserved + tracker components), spatial dimension, Q.  Any out pointer may be NULL. */
lbmk_status lbmk_system_info(const lbmk_system* sys, int* m_conserved, int* m_total, int* dim, int* Q);
/* Number of prescribed per-node coefficient fields of the system (0 for most). */
lbmk_status lbmk_system_aux_count(const lbmk_system* sys, int* n_aux);
/* Relaxation: conserved fields tau_k = 1/2 + tau_R[k]*dt; n = 1 (same for all) or
 * m_conserved.  Tracker fields relax at omega = 1/(g_tau+1) and use tau_grad = g_tau*dt in their flux and
 * source.  g_tau is ignored by tracker-free systems. */
lbmk_status lbmk_system_set_relaxation(lbmk_system* sys, const double* tau_R, int n, double g_tau);
/* Direct relaxation rates omega_k = 1/tau_k for all m_total components (n = 1 or m_total); overrides the
 * rule above.  omega = 0 gives pure streaming, omega = 1 the Lax-Friedrichs collapse. */
lbmk_status lbmk_system_set_omega(lbmk_system* sys, const double* omega, int n);
/* Reference state Q0 [m_total] of the shifted form (eq 2.23).  Default: zeros.  NSF3D / MHD3D require
 * zero reference momentum, magnetic field and trackers (LBMK_EUNSUPPORTED otherwise). */
lbmk_status lbmk_system_set_reference(lbmk_system* sys, const double* U0, int n);
/* Manufactured-solution forcing S_MMS of eq 4.1 for the augmented system, evaluated at
 * t_n + dt/2.  mms_id 0 = none, 1 = the system's manufactured fields.
 *   BURGERS2D {A};  EULER2D {};  SWE2D {A_h, A_u, h0};  ADR2D {};  NSF3D {U0, A_rho, rho0, p0};
 *   URF2D {} (eq SM5.4);  MAXWELL2D {} (eq SM5.5);  ALLENCAHN2D {} (eq SM5.8);
 *   INSE2D {U, rho0} (eq SM5.9);  ELASTICITY2D {} (eq SM5.6);
 *   NSF2D {} (eq SM5.10);  SWE2D_BATHY {h0, A_h, m0, A_m, A_zb, w_t} (eq SM5.3, bed L1198; w_t = frequency of the time factors);
 *   MHD2D {} (SM5.12 L1375-L1392).  HCNSF3D has none compiled in (its exact fields are truncated in the source, L1457). */
lbmk_status lbmk_system_set_mms(lbmk_system* sys, int mms_id, const double* mms_params, int n);
/* Collision operator.  LBMK_COLLISION_BGK (default) is eq 2.11, the operator the paper analyses and runs.  LBMK_COLLISION_TRT is
 * the two-relaxation-time operator the paper names as consuming the same equilibria unchanged, in its textbook
 * form: with ibar opposite to i and f+- = (f_i +- f_ibar)/2,
 *     f' = f_i - omega_plus (f+ - f_eq+) - omega_minus (f- - f_eq-) + w_i dt S,
 * omega_minus = the component's rate omega_k (f_eq- = w_i c_i.F/c_s^2 carries the flux, so the relaxation diffusion of eq 2.17 is
 * unchanged) and omega_plus from the magic parameter Lambda = (1/omega_plus - 1/2)(1/omega_minus - 1/2) (`magic` > 0; 1/4 is the
 * usual choice).  TRT runs on the two-lattice pull pattern with the node kernel, one launch per step (other options resolve
 * to these).  LBMK_COLLISION_REGULARIZED (the other operator L154 names): the non-equilibrium part is projected onto its first
 * moment before it is relaxed, f_neq,i -> w_i c_i.Pi/c_s^2 with Pi = sum_j c_j (f_j - f_eq,j); on D2Q5 / D3Q7 this keeps the
 * antisymmetric parts and removes the symmetric ones, so it runs as the two-rate kernel with omega_plus = 1 (`magic` ignored).
 * Not paper results: pinned by textbook properties and by the projection written out, tests/test_trt.py. */
enum { LBMK_COLLISION_BGK = 0, LBMK_COLLISION_TRT = 1, LBMK_COLLISION_REGULARIZED = 2 };
lbmk_status lbmk_system_set_collision(lbmk_system* sys, int collision, double magic);
/* A-priori bound on the physical wave speed max|eig sum n_a A_a| from the declared amplitudes (eq 2.20).
 * lbmk_grid_create rejects the grid with LBMK_ESUBCHAR if s_max/lambda > c_s.  0 = no declared bound. */
lbmk_status lbmk_system_set_wave_speed_bound(lbmk_system* sys, double s_max);
void lbmk_system_destroy(lbmk_system* sys);

/* ---- allocate a periodic or bounded grid ------------------------------------------------------------ */

/* nx, ny, nz >= 1 nodes (nz must be 1 for 2D systems); dx = node spacing; lambda = dx/dt the lattice
 * velocity (grid scaling).  The system is copied: later changes to *sys do not affect
 * the grid.  cuda_stream: a cudaStream_t.  With LBMK_DIRICHLET_MMS the outermost node layer is reset to
 * f_eq(Q_exact(x_b, t_n)) before every step and before readback (needs mms_id != 0; the paper defines no
 * boundary operator, PAPER.md:L504, L608 -- DESIGN.md reading A18). */
/* nx*ny*nz must be < 2^31 nodes (LBMK_EINVAL otherwise): node indices are 32-bit inside the kernels. */
lbmk_status lbmk_grid_create(const lbmk_system* sys, int nx, int ny, int nz, lbmk_bc bc, double dx, double lambda,
                             lbmk_precision precision, void* cuda_stream, lbmk_grid** out);
lbmk_status lbmk_grid_set_option(lbmk_grid* g, lbmk_option key, long long value);
lbmk_status lbmk_grid_get_option(const lbmk_grid* g, lbmk_option key, long long* value); /* resolved value */
/* Device bytes the grid needs (populations, trig tables, reduction scratch). */
lbmk_status lbmk_grid_workspace_bytes(const lbmk_grid* g, size_t* bytes);
/* device_ptr: DEVICE memory, 256-byte aligned, >= workspace_bytes; caller-owned, must outlive the grid. */
lbmk_status lbmk_grid_bind_workspace(lbmk_grid* g, void* device_ptr, size_t bytes);
void lbmk_grid_destroy(lbmk_grid* g);

/* ---- sub-domains and slabs -------------------------------------------------------- */

/* The grid is a sub-domain of a larger one: node (ix, iy, iz) sits at ((ix+ox) dx, (iy+oy) dx, (iz+oz) dx).  Only
 * explicit (x, t) dependence sees it (manufactured forcing and exact fields).  Before lbmk_grid_bind_workspace. */
lbmk_status lbmk_grid_set_origin(lbmk_grid* g, int ox, int oy, int oz);
/* Slab mode: the slowest axis (z in 3D, y in 2D) holds one GHOST plane at each end (plane 0 and plane n-1), the
 * planes between are the rank's own.  Forces the two-lattice pull pattern; the reductions (sub-characteristic
 * check, error norms) skip the ghost planes; lbmk_read_U still returns all planes (ghost values are meaningless).
 * lbmk_init_from_U must be given valid data on the ghost planes too (they are the neighbours' planes at t0).
 * After EVERY lbmk_step(g, 1) the face-crossing populations are exchanged with the two neighbours:
 *   lbmk_halo_pack   send_lo <- populations of the first own plane moving down, send_hi <- of the last own plane moving up
 *   (transport: the lower neighbour's send_hi is this rank's recv_lo, the upper neighbour's send_lo its recv_hi)
 *   lbmk_halo_unpack recv_lo -> lower ghost plane, recv_hi -> upper ghost plane.
 * Buffers: DEVICE pointers, lbmk_halo_bytes() each, layout [m_total][plane nodes] in the grid's storage type;
 * both calls are asynchronous on the grid's stream.  Before lbmk_grid_bind_workspace. */
lbmk_status lbmk_grid_set_slab(lbmk_grid* g, int enable);
lbmk_status lbmk_halo_bytes(const lbmk_grid* g, size_t* bytes);
lbmk_status lbmk_halo_pack(lbmk_grid* g, void* send_lo, void* send_hi);
lbmk_status lbmk_halo_unpack(lbmk_grid* g, const void* recv_lo, const void* recv_hi);
/* The same on another stream (a cudaStream_t; NULL = the grid's stream), so that the exchange can run beside the interior update. */
lbmk_status lbmk_halo_pack_on(lbmk_grid* g, void* send_lo, void* send_hi, void* cuda_stream);
lbmk_status lbmk_halo_unpack_on(lbmk_grid* g, const void* recv_lo, const void* recv_hi, void* cuda_stream);
/* Overlapped slab step (the exchange "overlapped with the interior update"):
 *   lbmk_step_slab(g)                     one step in three launches on the grid's stream: first own plane, last own plane,
 *                                         [boundary event], interior planes; ghost planes are not updated
 *   lbmk_stream_wait_boundary(g, s)       stream s waits for that boundary event (then: lbmk_halo_pack_on(.., s), transport,
 *                                         lbmk_halo_unpack_on(.., s) while the interior launch runs on the grid's stream)
 *   lbmk_grid_wait_stream(g, s)           the grid's stream waits for everything enqueued on s so far (before the next step).
 * The result equals lbmk_step(g, 1) + pack/transport/unpack bit for bit. */
lbmk_status lbmk_step_slab(lbmk_grid* g);
lbmk_status lbmk_stream_wait_boundary(lbmk_grid* g, void* cuda_stream);
lbmk_status lbmk_grid_wait_stream(lbmk_grid* g, void* cuda_stream);
/* Direct halo over peer memory: compute and transfer in ONE kernel.  The boundary-plane launches of lbmk_step_slab_peer store the
 * face-crossing populations, besides into this slab, straight into the ring neighbours' ghost planes: slot(-s) of the first own
 * plane into the lower neighbour's upper ghost plane, slot(+s) of the last own plane into the upper neighbour's lower ghost
 * plane -- peer device pointers (another GPU's memory over NVLink / NVSwitch mapped into this process, or another slab on the
 * same GPU).  No pack, no transport call, no unpack.
 *   lbmk_grid_population_buffers  this grid's two population buffers (DEVICE pointers into the bound workspace) and the first
 *                                 node of its upper ghost plane: what a neighbour needs to address this grid's ghost planes
 *   lbmk_grid_set_halo_peers      the neighbours' buffers: lower neighbour (f0, f1, first node of ITS upper ghost plane), upper
 *                                 neighbour (f0, f1; its lower ghost plane is plane 0).  All slabs of a ring step in lockstep, so
 *                                 buffer index b of this grid pairs with index b of its peers.
 *   lbmk_step_slab_peer           as lbmk_step_slab, boundary launches with the peer stores.  Ordering is the caller's: before the
 *                                 next step, this grid's stream must wait for BOTH neighbours' boundary events
 *                                 (lbmk_stream_wait_boundary(neighbour, this stream); across processes: an interprocess event).
 * The ghost slots receive exactly the values the boundary planes hold (the transfer is exact); the boundary planes themselves
 * are computed by the peer-store instantiation of the step kernel -- same arithmetic, but FMA contraction is nvcc's per kernel,
 * so against lbmk_step_slab + pack / transport / unpack nonlinear systems agree to rounding, linear ones bit for bit
 * (tests/test_gpu_slabs.py).  BGK with the node kernel only (LBMK_EUNSUPPORTED otherwise). */
lbmk_status lbmk_grid_population_buffers(const lbmk_grid* g, void** f0, void** f1, long long* upper_ghost_first_node);
lbmk_status lbmk_grid_set_halo_peers(lbmk_grid* g, void* lo_f0, void* lo_f1, long long lo_upper_ghost_first_node, void* hi_f0, void* hi_f1);
lbmk_status lbmk_step_slab_peer(lbmk_grid* g);

/* ---- initialise from U, step, read back U ------------------------------------------------------------ */

/* Step 0: all populations, conserved and tracker, at the (shifted) equilibrium of
 * U [m_total][nz][ny][nx] (fp64).  Sets step = 0, t = t0. */
lbmk_status lbmk_init_from_U(lbmk_grid* g, const double* U, int on_device, double t0);
/* Prescribed coefficient fields A [n_aux][nz][ny][nx] (fp64; stored in the grid's arithmetic type): SWE2D_BATHY the bed
 * slope (d_x z_b, d_y z_b) (eq 3.5); HCNSF3D the porosity and solid velocity (alpha, u_s) (eq 3.27).
 * Used by every later step until replaced (time-dependent fields: call again between steps; the paper takes explicit
 * (x, t) dependence at t_n + dt/2, L154).  Must be called before lbmk_init_from_U for systems with n_aux > 0
 * (LBMK_ESTATE otherwise); LBMK_EUNSUPPORTED for systems without.  Asynchronous for device pointers. */
lbmk_status lbmk_set_aux_fields(lbmk_grid* g, const double* A, int on_device);
/* Sets the populations directly (canonical layout below, fp64; stored as given minus the shift). */
lbmk_status lbmk_set_populations(lbmk_grid* g, const double* f, int on_device, double t0);
/* n_steps fused collide-and-stream steps (eq 2.11), asynchronous on the grid's stream. */
lbmk_status lbmk_step(lbmk_grid* g, int n_steps);
/* U_k = Q0_k + sum_i f*_k,i (eq 2.6; L312), returned as fp64 [m_total][nz][ny][nx].  Synchronises. */
lbmk_status lbmk_read_U(lbmk_grid* g, double* U_out, int on_device);
/* Canonical population state after the completed steps: f[k][i][node] = the (unshifted) population of
 * component k that sits at `node` and will next move along c_i -- independent of the storage pattern.
 * fp64 [m_total][Q][nz][ny][nx].  Synchronises. */
lbmk_status lbmk_read_populations(lbmk_grid* g, double* f_out, int on_device);
/* Completed steps and current time t0 + step*dt. */
lbmk_status lbmk_time(const lbmk_grid* g, long long* step, double* t);

/* ---- sub-characteristic check (eq 2.19-2.20; L329; eq 3.12) ------------------ */

/* Device max-reduction over the current state, in LATTICE units:
 *   out3[0] = max_x max_axis (|u_a| + c_a)/lambda   per-axis ceiling seen by D2Q5/D3Q7 streaming
 *   out3[1] = max_x (|u| + c)/lambda                isotropic bound over all directions n
 *   out3[2] = sqrt(kappa_L/g_tau)                   diffusive signal speed of the tracker-parent coupling
 * Returns LBMK_ESUBCHAR if max(out3[0], out3[1]) + out3[2] > c_s.  out3 is a HOST pointer (may be NULL). */
lbmk_status lbmk_check_subcharacteristic(lbmk_grid* g, double* out3);

/* ---- convergence study -------------------------------------------------------- */

/* Device reductions of the current state against the manufactured solution at the current time t0 + step*dt
 * (needs mms_id != 0, else LBMK_EUNSUPPORTED).  out: HOST pointer to [m_total][6] doubles,
 *   out[k] = { sum_x |e|, sum_x e^2, max_x |e|, sum_x |q|, sum_x q^2, max_x |q| },  e = U_k - Q_exact,k,  q = Q_exact,k,
 * all in fp64 (exact fields from their closed forms).  The paper's relative norms (L504) are
 * L1 = out[0]/out[3], L2 = sqrt(out[1]/out[4]), Linf = out[2]/out[5].  Synchronises. */
lbmk_status lbmk_error_norms(lbmk_grid* g, double* out);

/* The same norms for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): lbmk_error_norms stages its result through a stream-ordered device allocation, this entry point calls no
 * cudaMalloc / cudaFree / allocating routine at all.  out_device: DEVICE pointer to [m_total][6] doubles, layout as above.
 * The work -- a Dirichlet frame refresh on bounded grids, then two kernels -- is enqueued on the grid's stream and NOT synchronised.
 * The reduction is a fixed two-pass tree: one record [m_total][6] per 4096 consecutive nodes, records combined in index order,
 * so the result is bit-reproducible and independent of the SM count (lbmk_error_norms accumulates with atomics; the sums of the
 * two agree to rounding, the maxima exactly).  The records live in a static device array of LBMK_NOALLOC_SCRATCH_BYTES that
 * every GPU that loads the library holds until exit; a grid that needs more --
 *     ceil(nx*ny*nz / 4096) * m_total * 48 bytes   (all BASELINE.json configs fit: c4 256^3 needs 3.3 MB)
 * -- is refused with LBMK_EINVAL and a message naming both sizes (checked before anything else about the grid's state).
 * ALL calls on one device share that array: two such calls that may overlap on the GPU (different streams) race; serialise them. */
#define LBMK_NOALLOC_SCRATCH_BYTES (4 * 1024 * 1024)
lbmk_status lbmk_error_norms_noalloc(lbmk_grid* g, double* out_device);

/* ---- test hooks ------------------------------------------------------------------------------------- */

/* For every node x: linear index of the node whose post-collision population `dir` arrives at x, i.e.
 * wrap(x - c_dir), computed on the device by the index functions the step kernels use.  int64
 * [nz][ny][nx]; bit-exact against the oracle's table. */
lbmk_status lbmk_stream_index_map(lbmk_grid* g, int dir, long long* src_index_out, int on_device);
/* Build-time generator check (Alg 2.1).  gen/cascade.py derives the augmented
 * system (trackers, chain rule, lattice scaling) of every system of this library from the declared conservation laws and emits
 * csrc/cascade_generated.cuh -- conserved-field trackers + chain rule (ADR, Allen-Cahn, INSE, NSF 2D, MHD 2D), derived-parent
 * trackers (NSF 3D), combination trackers (HCNSF's symmetric gradient, MHD 3D's curl), and the tracker-free systems.
 *   lbmk_generated_flux   evaluates the emitted code on the HOST (no GPU needed) at one state: U [m_total], A [n_aux] or NULL,
 *                         params as for lbmk_system_create; F_out [m_total][3] lattice flux (dt/dx) Phi, S_out [m_total] lattice
 *                         source dt S, trackers in lattice units.
 *   lbmk_flux_selfcheck   on the device, for every node of the grid's current state: the hand-written delta-form flux/source the
 *                         step kernels use against the emitted plain form, in fp64; *max_rel_diff = the largest difference
 *                         relative to the node's largest flux/source entry (rounding level when the two derivations agree). */
lbmk_status lbmk_generated_flux(lbmk_system_id id, const double* U, const double* A, const double* params, int n_params,
                                double dx, double lambda, double g_tau, double* F_out, double* S_out);
lbmk_status lbmk_flux_selfcheck(lbmk_grid* g, double* max_rel_diff);
/* Lattice constants as the kernels use them: c [Q][3] int, w [Q], c_s^2.  Host pointers. */
lbmk_status lbmk_lattice_constants(lbmk_lattice lattice, int* c, double* w, double* cs2);
/* Relaxation rates omega_k [m_total] the grid uses.  Host pointer. */
lbmk_status lbmk_grid_omega(const lbmk_grid* g, double* omega_out);
/* TRT: rates omega_plus,k [m_total] of the symmetric parts (equal to omega_k for BGK).  Host pointer. */
lbmk_status lbmk_grid_omega_plus(const lbmk_grid* g, double* omega_out);
/* Kernel launches enqueued by this grid so far (bench.py's gpu_launches). */
lbmk_status lbmk_grid_launch_count(const lbmk_grid* g, long long* launches);
/* CUDA-event time, in milliseconds, of the collide-and-stream kernels of the most recent lbmk_step call
 * (first kernel start to last kernel end, on the grid's stream).  Synchronises. */
lbmk_status lbmk_last_step_ms(lbmk_grid* g, float* ms);

/* Message of the last failure on this grid (g != NULL) or in this thread's system calls (g == NULL). */
const char* lbmk_last_error(const lbmk_grid* g);
const char* lbmk_version(void);

/* Streaming-bandwidth probe: a plain device copy of `bytes` bytes (read + write) repeated `reps` times on
 * `cuda_stream`; *gbs receives (2*bytes*reps)/time.  The like-for-like roofline denominator, cf. the
 * paper's BabelStream Triad peak.  src/dst: device pointers, 16-byte aligned. */
lbmk_status lbmk_copy_bandwidth(void* dst, const void* src, size_t bytes, int reps, void* cuda_stream, double* gbs);

#ifdef __cplusplus
}
#endif
#endif /* LBMK_H */
