// ops.h -- type-erased per-system entry points: the seam between the C-ABI (lbmk_api.cu, host logic) and
// the templated kernels (one translation unit per system, sys_*.cu, instantiating ops_impl.cuh).
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"

namespace lbmk {

enum { PREC_F64 = 0, PREC_F32 = 1 };
enum { PATTERN_PULL2 = 1, PATTERN_AA = 2 };
enum { KERNEL_NODE = 1, KERNEL_ROW = 2, KERNEL_TWOPASS = 3 };
enum { STEPPING_LAUNCH = 1, STEPPING_PERSISTENT = 2, STEPPING_CLUSTER = 3, STEPPING_RESIDENT = 4 };

struct GridCore {
    int nx, ny, nz;
    long long n;
    int prec;             // PREC_F64 / PREC_F32 (storage and arithmetic type R)
    int bc;               // 0 periodic, 1 Dirichlet-MMS frame
    int pattern, kernel;
    int mms_id;
    cudaStream_t stream;
    void* f[2];           // population buffers; f[1] == nullptr for the in-place AA pattern
    int cur;              // PULL2: which buffer holds the current state
    int pending;          // PULL2: storage is post-collision, the stream is pending (kernels.cuh GATHER_PULL)
    long long step;       // completed steps
    double t0, dt;
    void* tab[3];         // per-axis trig tables in R, [entry][index]
    void* coef;           // per-row forcing coefficients in R: 2 buffers x [coef_B steps][nz*ny][nc]
    int coef_B;           // steps per coefficient batch (one pre-kernel launch fills a batch)
    cudaStream_t aux;     // the pre-kernel of batch j+1 runs here while the steps of batch j run on `stream`
    cudaEvent_t ev_entry, ev_coef[2], ev_free[2];
    bool coef_used[2];
    double* feq0;         // [M*Q] reference equilibrium (fp64)
    unsigned long long* red;   // [4] reduction scratch
    unsigned int* bar;    // PERSISTENT_MAX_BLOCKS "steps done" flags of the persistent kernel, one per block (zeroed before each launch)
    void* aux_buf;        // prescribed coefficient fields in R, [n_aux][aux_stride]
    long long aux_stride;
    bool aux_set;
    int collision;        // 0 BGK, 1 TRT (two-lattice pull, node kernel, one launch per step)
    int stepping;         // STEPPING_LAUNCH: one launch per step; STEPPING_PERSISTENT: one cooperative launch per batch of steps
    int num_sms;          // cudaDevAttrMultiProcessorCount of the current device
    void* peer_f[2][2];   // direct halo: [lo|hi][buffer index] population buffers of the ring neighbours (peer device memory)
    long long peer_node0[2];   // first node of the ghost plane to fill at the lower / upper neighbour
    bool peers_set;
    long long persistent_launches;   // cooperative launches so far (diagnostic)
    KParams<double> Pd;   // parameters in fp64 (host logic, fp64 kernels, readback)
    KParams<float> Pf;    // same, rounded to fp32 (fp32 kernels)
    MmsHostArgs mh;
    long long launches;
};

struct SysOps {
    int id, D, M, MC;
    bool has_mms;
    int nt, nax[3];       // time scalars and table entries per axis of the manufactured solution
    int nc;               // per-row forcing coefficients (multiple of 4; 0 without manufactured solution)
    int n_aux;            // prescribed per-node coefficient fields
    bool linear;          // single-product flux entries: bits independent of the kernel (AUTO may then pick the cluster kernel)
    // all return cudaError_t of the last launch / API call
    cudaError_t (*fill_tables)(GridCore&);                 // host fp64 -> device R tables (synchronous copy on the stream)
    cudaError_t (*reference_equilibrium)(GridCore&);
    cudaError_t (*init_from_U)(GridCore&, const double* U_dev);
    cudaError_t (*set_f)(GridCore&, const double* f_dev);
    cudaError_t (*step)(GridCore&, int n_steps);
    // one step in up to 3 launches: nodes [a0,a1) and [b0,b1) first (the slab's boundary planes), then `ev` is recorded on
    // the stream, then [c0,c1) (the interior); empty ranges are skipped
    cudaError_t (*step_ranges)(GridCore&, const long long* ranges6, cudaEvent_t ev, int peer);   // peer: boundary ranges also store into the neighbours' ghost planes
    cudaError_t (*set_aux)(GridCore&, const double* A_dev);
    cudaError_t (*read_U)(GridCore&, double* U_dev);
    cudaError_t (*read_f)(GridCore&, double* f_dev);
    cudaError_t (*max_wave_speed)(GridCore&, double* out3_host);
    cudaError_t (*error_norms)(GridCore&, double* out_dev /*[M][6], zeroed here*/);
    bool (*row_kernel_supported)(const GridCore&);
    bool (*cluster_supported)(const GridCore&);
    bool has_generated;   // gen/cascade.py emits this system: lbmk_flux_selfcheck is available
    cudaError_t (*flux_selfcheck)(GridCore&, double g_tau, double* out_host);
    bool (*resident_supported)(const GridCore&);
    // node ranges of init_from_U / read_U (host buffers go through fixed-size staging chunks): U holds [node0, node1), planes ustride apart
    cudaError_t (*init_range)(GridCore&, const double* U, long long ustride, long long node0, long long node1);
    cudaError_t (*read_range)(GridCore&, double* U, long long ustride, long long node0, long long node1);
    cudaError_t (*frame_now)(GridCore&);            // Dirichlet frame refresh before a readback
    // error norms through caller-independent scratch [ceil(n / NORM_RECORD_NODES)][M][6] doubles, into out_dev [M][6]; nothing allocated
    cudaError_t (*error_norm_records)(GridCore&, double* scratch, double* out_dev);
     // one population copy fits the shared memory of all SMs (kernels.cuh collide_stream_resident)
};

const SysOps* ops_advection2d();
const SysOps* ops_burgers2d();
const SysOps* ops_swe2d();
const SysOps* ops_euler2d();
const SysOps* ops_adr2d();
const SysOps* ops_nsf3d();
const SysOps* ops_mhd3d();
const SysOps* ops_urf2d();
const SysOps* ops_maxwell2d();
const SysOps* ops_allencahn2d();
const SysOps* ops_inse2d();
const SysOps* ops_elasticity2d();
const SysOps* ops_nsf2d();
const SysOps* ops_swe2d_bathy();
const SysOps* ops_hcnsf3d();
const SysOps* ops_mhd2d();

}  // namespace lbmk
