// common.cuh -- lattice constants, kernel parameter block and index functions of the CUDA path.
//
// Lattices: Table SM1.  D2Q5: w = 1/3, 1/6, c_s^2 = 1/3; D3Q7: w = 1/4, 1/8,
// c_s^2 = 1/4.  Direction order (free choice, reading A10): 0 rest; 1:+x 2:-x 3:+y 4:-y 5:+z 6:-z;
// opposite(i) pairs (1,2), (3,4), (5,6).  On both lattices w_i / c_s^2 = 1/2 for the moving directions.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

#include "mms_generated.cuh"

namespace lbmk {

// Components whose populations the per-launch two-lattice kernel with forcing keeps in a shared-memory park instead of registers
// (kernels.cuh collide_core); specialised per system in systems.cuh
template <class Sys> struct ParkCount { static constexpr int value = 0; };

constexpr int NORM_RECORD_NODES = 4096;        // nodes per partial record of the two-pass error norms (kernels.cuh, lbmk_error_norms_noalloc)
constexpr int PERSISTENT_MAX_BLOCKS = 2048;   // "steps done" flags of the persistent kernel: one per block,
constexpr int FLAG_STRIDE = 32;              // each in its own 128-byte line (32 words apart)


constexpr int MAXM = 20;   // largest compiled-in system has 18 components

template <int D> struct Lattice;
template <> struct Lattice<2> {
    static constexpr int Q = 5;
    static constexpr double w0 = 1.0 / 3.0, w1 = 1.0 / 6.0, cs2 = 1.0 / 3.0;
};
template <> struct Lattice<3> {
    static constexpr int Q = 7;
    static constexpr double w0 = 1.0 / 4.0, w1 = 1.0 / 8.0, cs2 = 1.0 / 4.0;
};

// Weights in the arithmetic type R.  The moving weight is w1 rounded to R; the rest weight is taken as 1 - 2D*w1 IN R, so
// that the weights sum to exactly 1 in the arithmetic the kernels run in.  In fp32 on D2Q5, float(1/3) + 4*float(1/6) =
// 1 + 3e-8: with the plainly rounded w0 every collision would multiply the (shifted) zeroth moment by 1 + omega*3e-8 -- a
// systematic drift, linear in the step count (3e-3 of the fluctuation after 1.4e5 steps), not rounding noise.  1 - 4*w1 is
// exact (Sterbenz), differs from 1/3 by 2e-8 (inside fp32 rounding of the oracle's value) and conserves exactly.  D3Q7's
// 1/4, 1/8 and the fp64 path (1/3 + 4/6 == 1 in double rounding) are unaffected.
template <int D, class R> __host__ __device__ constexpr R weight1() { return R(Lattice<D>::w1); }
template <int D, class R> __host__ __device__ constexpr R weight0() {
    return std::is_same<R, float>::value ? R(1) - R(2 * D) * R(Lattice<D>::w1) : R(Lattice<D>::w0);
}

__host__ __device__ constexpr int opposite(int i) { return i == 0 ? 0 : (((i - 1) ^ 1) + 1); }
// c_i component along axis a (0 x, 1 y, 2 z)
__host__ __device__ constexpr int cvel(int i, int a) { return (i == 0 || (i - 1) / 2 != a) ? 0 : (((i - 1) & 1) ? -1 : +1); }

// Kernel parameter block (passed by value).  R = arithmetic/storage type of the path.
template <class R>
struct KParams {
    int nx, ny, nz;
    long long n;            // nodes
    int ox, oy, oz;         // node (ix, iy, iz) sits at ((ix+ox) dx, (iy+oy) dx, (iz+oz) dx): sub-domain of a larger grid
    int ghost;              // 1: slab with one ghost plane at each end of the slowest axis (skipped by the reductions)
    R omega[MAXM];          // relaxation rate per component; TRT: rate of the antisymmetric parts
    R omega_p[MAXM];        // TRT only: rate of the symmetric parts (from the magic parameter)
    R ref[MAXM];            // reference state Q0 of eq (2.23); zeros in the unshifted fp64 form
    R par[8];               // physical parameters of the system
    R cst[8];               // host-derived reference constants (u0, p0, E0+p0, T0, ...), see systems.cuh
    R il;                   // dt/dx = 1/lambda
    R dL;                   // dt/dx^2: physical diffusivity -> lattice diffusivity
    R inv_gtau;             // 1/g_tau
    R dt;
    // manufactured forcing (eq 4.1): time scalars at t_n + dt/2 and per-axis tables [entry][index]
    MmsArgs<R> mms;
    R T[8];
    const R* tabX;
    const R* tabY;
    const R* tabZ;
    const R* coef;          // per-row forcing coefficients [nz*ny][Mms::NC], rewritten before every step
    // prescribed per-node coefficient fields (bed slope of eq 3.5): aux[a * aux_stride + node], in R
    const R* aux;
    long long aux_stride;
    // node range [node0, node1) a step launch updates (whole grid: 0, n); block b starts at node0 + b*BLOCK
    long long node0, node1;
    // direct halo (slabs, peer stores): this step's destination buffers of the lower / upper ring neighbour (peer device
    // memory: another GPU over NVLink, or another slab on this GPU) and the first node of the ghost plane to fill there
    R* peer_lo;
    R* peer_hi;
    long long peer_lo_node0, peer_hi_node0;
    long long plane_nodes;  // nodes per plane of the slab axis
    long long last_own0;    // first node of the last own plane
};

// number of prescribed coefficient fields of a system: Sys::NA where declared, else 0
template <class S, class = void> struct AuxCount { static constexpr int value = 0; };
template <class S> struct AuxCount<S, std::void_t<decltype(S::NA)>> { static constexpr int value = S::NA; };
// systems whose flux entries are single products (Sys::LINEAR): their results do not depend on which kernel computed them
template <class S, class = void> struct IsLinear { static constexpr bool value = false; };
template <class S> struct IsLinear<S, std::void_t<decltype(S::LINEAR)>> { static constexpr bool value = S::LINEAR; };

struct NodeIdx { int ix, iy, iz; };

__device__ __forceinline__ NodeIdx decompose(long long node, int nx, int ny) {
    // nx*ny*nz < 2^31 is checked at grid creation: 32-bit unsigned divisions (no 64-bit division subroutine)
    NodeIdx p;
    const unsigned nd = (unsigned)node;
    const unsigned row = nd / (unsigned)nx;
    p.ix = (int)(nd - row * (unsigned)nx);
    const unsigned iz = row / (unsigned)ny;
    p.iz = (int)iz;
    p.iy = (int)(row - iz * (unsigned)ny);
    return p;
}

// Element offset from `node` to the periodic neighbour node - c_i (the node a pull along direction i
// reads from), i.e. wrap(x - c_i) - x in linear index space.  The ONE place the streaming index map is
// defined on the device: the step kernels, the readback gathers and lbmk_stream_index_map all call it.
__device__ __forceinline__ long long pull_offset(int i, const NodeIdx& p, int nx, int ny, int nz) {
    switch (i) {
        case 1: return p.ix == 0 ? (long long)(nx - 1) : -1LL;
        case 2: return p.ix == nx - 1 ? -(long long)(nx - 1) : 1LL;
        case 3: return p.iy == 0 ? (long long)(ny - 1) * nx : -(long long)nx;
        case 4: return p.iy == ny - 1 ? -(long long)(ny - 1) * nx : (long long)nx;
        case 5: return p.iz == 0 ? (long long)(nz - 1) * nx * ny : -(long long)nx * ny;
        case 6: return p.iz == nz - 1 ? -(long long)(nz - 1) * nx * ny : (long long)nx * ny;
        default: return 0LL;
    }
}
// Offset to node + c_i (push target): the pull offset of the opposite direction.
__device__ __forceinline__ long long push_offset(int i, const NodeIdx& p, int nx, int ny, int nz) {
    return pull_offset(opposite(i), p, nx, ny, nz);
}

// Population storage: tiled structure of arrays.  Nodes are grouped, in linear index order, into tiles of TILE
// consecutive nodes (x fastest, so a tile is an x-row segment); within a tile the M*Q population planes are
// stored one after the other, TILE elements each:
//     element(plane, node) = (node / TILE) * (M*Q*TILE) + plane * TILE + node % TILE .
// A thread block therefore streams ONE contiguous M*Q*TILE*sizeof(R) chunk per direction (c4: 60 KB) instead
// of M*Q segments from planes a whole grid apart, and -- the point for the step kernels -- the plane offset
// is a compile-time constant: every access is [per-direction base pointer + immediate], with no address
// arithmetic per population.  The last tile is padded (allocation = n_tiles * TILE nodes).
constexpr int LOG_TILE = 7, TILE = 1 << LOG_TILE;
__host__ __device__ __forceinline__ long long tile_off(long long node, int MQ) {
    return (node >> LOG_TILE) * ((long long)MQ << LOG_TILE) + (node & (TILE - 1));
}

// Compile-time loop
template <int I, int N, class F>
__host__ __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(static_cast<F&&>(f));
    }
}

}  // namespace lbmk
