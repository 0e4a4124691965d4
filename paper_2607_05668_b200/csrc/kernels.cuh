// kernels.cuh -- the collide-and-stream step (one node per thread, direct loads) and its service kernels.
//
// Population storage: tiled structure of arrays, element(k*Q + i, node) = tile_off(node) + (k*Q + i)*TILE
// (common.cuh).
// Step per node (eq 2.6 / 2.7 / 2.11 of the paper):
//   gather f_k,i  ->  dQ_k = sum_i f_k,i  ->  dF_k, s_k (systems.cuh; + manufactured forcing at t_n + dt/2)
//   ->  f' = f - omega_k (f - w_i (dQ_k + c_i.dF_k/c_s^2)) + w_i s_k  ->  scatter.
// Because c_i are the axis unit vectors and w_i/c_s^2 = 1/2 for them, the relaxation reads
//   rest:   f' = (1-omega) f + w0 (omega dQ + s)
//   +-a:    f' = (1-omega) f + w1 (omega dQ + s) +- (omega/2) dF_a .
// Streaming patterns (MODE).  Canonical state after n steps: slot i at x holds the population that arrived
// at x along c_i (what the oracle's array holds after its stream).  Storage states (GATHER_*):
//   two-lattice pull: the first step after init is LOCAL (read slot i at x of `src`, collide, write slot i at
//     x of `dst`); the storage is then post-collision with the stream pending (GATHER_PULL: the canonical
//     population (i, x) sits in slot i at x - c_i), and every further step is PULL2: read slot i at x - c_i,
//     collide, write slot i at x.  n steps = n kernels; the last stream is done by whoever reads the state.
//   AA is in place: the even step reads slot i at x and writes slot opp(i) at x (GATHER_AA_ODD: canonical
//     (i, x) sits in slot opp(i) at x - c_i), the odd step reads that and writes slot i at x + c_i, which is
//     canonical again.
#pragma once
#include <cooperative_groups.h>

#include "systems.cuh"

namespace lbmk {

enum { MODE_PULL2 = 0, MODE_AA_EVEN = 1, MODE_AA_ODD = 2, MODE_LOCAL = 3 };
enum { GATHER_CANON = 0, GATHER_AA_ODD = 1, GATHER_PULL = 2 };

template <class Sys> __host__ __device__ constexpr bool has_mms() { return !std::is_void<typename Sys::Mms>::value; }
template <class Sys, bool = has_mms<Sys>()> struct MmsNC { static constexpr int value = 4; };
template <class Sys> struct MmsNC<Sys, true> { static constexpr int value = Sys::Mms::NC; };
// Row coefficients are staged in shared memory (cp.async + one bar.sync per segment) only when there are enough of them to
// pay for the barrier: measured on c2 (12 coefficients) the warp-uniform global loads are 0.6 us per step faster, on c4 (108)
// the staged copy wins.
constexpr int STAGE_MIN_NC = 48;

// per-node manufactured forcing: the x-table entries of this node and the coefficients of its (y, z) row
// (mms_generated.cuh source_row; the row table is filled by mms_row_coeffs_kernel).  SH: `c` is the block's
// shared-memory copy of its row, otherwise `c` is this step's coefficient table in global memory.
template <class Sys, class R, bool SH>
__device__ __forceinline__ void mms_node(const KParams<R>& P, const NodeIdx& p, const R* c, R (&s)[Sys::M]) {
    if constexpr (has_mms<Sys>()) {
        using G = typename Sys::Mms;
        R X[G::NX > 0 ? G::NX : 1];
#pragma unroll
        for (int e = 0; e < G::NX; ++e) X[e] = __ldg(P.tabX + e * P.nx + p.ix);
        if (!SH) c = c + (size_t)(p.iz * P.ny + p.iy) * G::NC;      // c = this step's coefficient table
        G::template source_row<R, SH>(c, X, s);
    }
}

// When nx is a multiple of the block size a thread block lies inside ONE (y, z) row: its NC coefficients are
// copied to shared memory with 16-byte cp.async issued BEFORE the population gather, so that the forcing reads
// them with short-latency LDS.128 instead of chains of L2 round trips queued behind the gather.
template <class R>
__device__ __forceinline__ void cp_async16(R* smem_dst, const R* gmem_src) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem_src) : "memory");
}
template <class R>
__device__ __forceinline__ void cp_async4(R* smem_dst, const R* gmem_src) {
    static_assert(sizeof(R) == 4, "4-byte copy");
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gmem_src) : "memory");
}
template <> __device__ __forceinline__ void cp_async4<double>(double*, const double*) {}     // never selected (PARK is fp32 only)
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Row coefficients of the forcing for `nb` consecutive steps: one thread per (step, (y, z) row), fp64 from the
// closed forms (no tables), stored in R as coef[b][row][NC].  Step b is forced at its temporal midpoint
// t_first + b dt + dt/2.  ~1e3 flops x ny*nz threads per step: negligible next to the step,
// and it runs on the auxiliary stream under the previous batch's steps.
template <class Sys, class R>
__global__ void __launch_bounds__(128)
mms_row_coeffs_kernel(R* __restrict__ coef, int ny, int nz, int oy, int oz, int nb, double t_first, double dt,
                      const __grid_constant__ MmsHostArgs mh, const __grid_constant__ MmsArgs<double> ma) {
    if constexpr (has_mms<Sys>()) {
        using G = typename Sys::Mms;
        const int rows = ny * nz;
        const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (id >= (long long)rows * nb) return;
        const int b = (int)(id / rows), row = (int)(id - (long long)b * rows);
        const int iz = row / ny, iy = row - iz * ny;
        double T[8], Y[8], Z[8];
        const double t_n = t_first + (double)b * dt;
        G::time_scalars(t_n + 0.5 * dt, mh, T);
        G::axis_row(1, (iy + oy) * mh.dx, mh, Y);
        if (G::NZ > 0) G::axis_row(2, (iz + oz) * mh.dx, mh, Z);
        G::template row_coeffs<double, R>(ma, T, Y, Z, coef + (size_t)id * G::NC);
    }
}

// BGK relaxation of one component's Q populations, in registers (f[0] rest, f[1+2a] = +a, f[2+2a] = -a)
template <int D, class R>
__device__ __forceinline__ void relax(R (&f)[2 * D + 1], R omega, R dQ, const R (&F)[D], R S) {
    using L = Lattice<D>;
    const R keep = R(1) - omega;
    const R A = omega * dQ + S;
    const R a0 = weight0<D, R>() * A, a1 = weight1<D, R>() * A;
    const R hw = R(0.5) * omega;
    f[0] = keep * f[0] + a0;
#pragma unroll
    for (int a = 0; a < D; ++a) {
        const R h = hw * F[a];
        f[1 + 2 * a] = keep * f[1 + 2 * a] + (a1 + h);
        f[2 + 2 * a] = keep * f[2 + 2 * a] + (a1 - h);
    }
}

// Two-relaxation-time relaxation (PAPER.md:L154 names TRT as an operator that consumes the same equilibria; textbook form):
// symmetric parts s = (f_+a + f_-a)/2 relax to w1 dQ at omega_p, antisymmetric parts d = (f_+a - f_-a)/2 relax to
// w1 c.F/c_s^2 = F_a/2 at omega (the flux-carrying rate, so the relaxation diffusion of eq 2.17 is unchanged); source as in BGK.
template <int D, class R>
__device__ __forceinline__ void relax_trt(R (&f)[2 * D + 1], R omega_p, R omega_m, R dQ, const R (&F)[D], R S) {
    const R keep_p = R(1) - omega_p, keep_m = R(1) - omega_m;
    const R A = omega_p * dQ + S;
    const R a0 = weight0<D, R>() * A, a1 = weight1<D, R>() * A;
    const R hw = R(0.5) * omega_m;
    f[0] = keep_p * f[0] + a0;
#pragma unroll
    for (int a = 0; a < D; ++a) {
        const R s = R(0.5) * (f[1 + 2 * a] + f[2 + 2 * a]), d = R(0.5) * (f[1 + 2 * a] - f[2 + 2 * a]);
        const R s1 = keep_p * s + a1, d1 = keep_m * d + hw * F[a];
        f[1 + 2 * a] = s1 + d1;
        f[2 + 2 * a] = s1 - d1;
    }
}

// Pointer qualifiers of the step kernels: the two-lattice modes of the per-launch kernels read one buffer and write the
// other, so both carry __restrict__ (loads may use the non-coherent path and move freely across the stores); the
// in-place AA modes are launched with src == dst, where __restrict__ would be a false promise -- plain pointers there.
// COHERENT (the persistent multi-step kernel): a buffer written in one step is read in the next step of the SAME launch,
// so neither const __restrict__ (-> ld.global.nc) is allowed; plain pointers, ordered by the grid barrier.
template <class R, int MODE, bool COHERENT = false> struct StepPtr { using Src = const R* __restrict__; using Dst = R* __restrict__; };
template <class R, bool C> struct StepPtr<R, 1 /*MODE_AA_EVEN*/, C> { using Src = const R*; using Dst = R*; };
template <class R, bool C> struct StepPtr<R, 2 /*MODE_AA_ODD*/, C> { using Src = const R*; using Dst = R*; };
template <class R> struct StepPtr<R, 0 /*MODE_PULL2*/, true> { using Src = const R*; using Dst = R*; };
template <class R> struct StepPtr<R, 3 /*MODE_LOCAL*/, true> { using Src = const R*; using Dst = R*; };

// prescribed coefficient fields of `node` into the system's context (systems with NA > 0 only)
template <class Sys, class R>
__device__ __forceinline__ void load_aux(typename Sys::Ctx& ctx, const KParams<R>& P, long long node) {
    constexpr int NA = AuxCount<Sys>::value;
    if constexpr (NA > 0) {
        R A[NA];
#pragma unroll
        for (int a = 0; a < NA; ++a) A[a] = __ldg(P.aux + a * P.aux_stride + node);
        Sys::set_aux(ctx, A);
    }
}

// a3-a6 of ONE node, in registers: moments, system algebra, equilibrium + BGK relaxation component by component; `store(K, f_k)`
// is called with the Q post-collision populations of component k as soon as they exist (so their registers die early).
// Shared by every step kernel -- one definition of the arithmetic, hence identical bits whatever the storage.
// PARK > 0: the populations of the LAST `PARK` components are not in f[][] but in the thread's slots of a shared-memory park
// (element (kk*Q + i)*PSTRIDE of `park`, filled by cp.async during the gather): they are read for the moment sum and again
// right before their relaxation, so they never occupy registers across the collision of the other components.
template <class Sys, class R, bool MMS, bool TRT = false, int PARK = 0, int PSTRIDE = 1, class Store>
__device__ __forceinline__ void collide_core(R (&f)[Sys::M][2 * Sys::D + 1], typename Sys::Ctx& ctx, const KParams<R>& P,
                                             const R (&smms)[Sys::M], const volatile R* park, Store&& store) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    R dQ[M];
#pragma unroll
    for (int k = 0; k < M; ++k) {
        if (PARK > 0 && k >= M - PARK) {
            R s = park[((k - (M - PARK)) * Q) * PSTRIDE];
#pragma unroll
            for (int i = 1; i < Q; ++i) s += park[((k - (M - PARK)) * Q + i) * PSTRIDE];
            dQ[k] = s;
        } else {
            R s = f[k][0];
#pragma unroll
            for (int i = 1; i < Q; ++i) s += f[k][i];
            dQ[k] = s;
        }
    }
    Sys::setup(ctx, dQ, P);
    static_for<0, M>([&](auto K) {
        constexpr int k = decltype(K)::value;
        R F[D], S;
        Sys::template flux<k>(ctx, dQ, P, F, S);
        if constexpr (PARK > 0 && k >= M - PARK) {
#pragma unroll
            for (int i = 0; i < Q; ++i) f[k][i] = park[((k - (M - PARK)) * Q + i) * PSTRIDE];
        }
        if constexpr (MMS) S += smms[k];
        if constexpr (TRT) relax_trt<D, R>(f[k], P.omega_p[k], P.omega[k], dQ[k], F, S);
        else relax<D, R>(f[k], P.omega[k], dQ[k], F, S);
        store(K, f[k]);
    });
}

// ------------------------------------------------------------------------------------------------ step
// The update of ONE node by ONE thread (a1-a7).  `first` = first node of this thread block's BLOCK-node segment,
// coef_s = the block's shared-memory slot for its row's forcing coefficients, coef = this step's coefficient table.
// Called by the per-launch kernel (one segment per block) and by the persistent kernel (segments in a loop): the
// same code, hence the same bits.
template <class Sys, class R, int MODE, bool MMS, int BLOCK, bool COHERENT, bool TRT = false, bool PEER = false, int PARK = 0>
__device__ __forceinline__ void node_step(typename StepPtr<R, MODE, COHERENT>::Src src, typename StepPtr<R, MODE, COHERENT>::Dst dst,
                                          const KParams<R>& P, const R* coef, long long first, R* coef_s, R* park_s = nullptr) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    static_assert(PARK == 0 || ((MODE == MODE_PULL2 || MODE == MODE_LOCAL) && !COHERENT && sizeof(R) == 4), "parked components: two-lattice fp32 per-launch kernel");
    const long long node = first + threadIdx.x;
    constexpr int NCs = MMS ? MmsNC<Sys>::value : 4;
    // kernel-uniform: a block lies inside one (y, z) row; then every segment is full (n and node0 are multiples of BLOCK)
    const bool staged = MMS && NCs >= STAGE_MIN_NC && (P.nx % BLOCK == 0) && (P.node0 % BLOCK == 0);
    if constexpr (MMS) {
        if (staged) {
            const unsigned row = (unsigned)(first / P.nx);
            constexpr int per = 16 / sizeof(R);
            if (threadIdx.x < NCs / per) cp_async16(coef_s + per * threadIdx.x, coef + (size_t)row * NCs + per * threadIdx.x);
            cp_async_commit();
        }
    }
    if (node >= P.node1) return;
    const NodeIdx p = decompose(node, P.nx, P.ny);
    // gather addresses: one 64-bit pointer per direction (the source node's slot in its tile); the plane offset
    // (k*Q + slot)*TILE is a compile-time constant, so every access is [pointer + immediate]
    const R* sp[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i)
        sp[i] = src + tile_off(node + ((MODE == MODE_AA_EVEN || MODE == MODE_LOCAL) ? 0LL : pull_offset(i, p, P.nx, P.ny, P.nz)), M * Q);
    R* const dp = dst + tile_off(node, M * Q);
    // PEER (boundary planes of a slab): the face-crossing populations are ALSO stored straight into the ring neighbour's ghost
    // plane -- slot(-s) of the first own plane into the lower neighbour's upper ghost plane, slot(+s) of the last own plane into
    // the upper neighbour's lower ghost plane -- so compute and halo transfer are one kernel over peer memory
    R* plo = nullptr;
    R* phi = nullptr;
    if constexpr (PEER) {
        if (node >= P.plane_nodes && node < 2 * P.plane_nodes) plo = P.peer_lo + tile_off(P.peer_lo_node0 + (node - P.plane_nodes), M * Q);
        if (node >= P.last_own0 && node < P.last_own0 + P.plane_nodes) phi = P.peer_hi + tile_off(P.peer_hi_node0 + (node - P.last_own0), M * Q);
    }

    R f[M][Q];
#pragma unroll
    for (int k = 0; k < M; ++k)
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            const int slot = (MODE == MODE_AA_ODD) ? opposite(i) : i;
            if constexpr (PARK > 0) {
                if (k >= M - PARK) {        // no register destination: asynchronous copy into this thread's slot of the park
                    cp_async4(park_s + ((k - (M - PARK)) * Q + i) * BLOCK + threadIdx.x, sp[i] + (k * Q + slot) * TILE);
                    continue;
                }
            }
            // persistent kernel: the line may sit stale in this SM's L1 from two steps ago -> read at L2 (ld.global.cg)
            f[k][i] = COHERENT ? __ldcg(sp[i] + (k * Q + slot) * TILE) : sp[i][(k * Q + slot) * TILE];
        }
    if constexpr (PARK > 0) cp_async_commit();
    typename Sys::Ctx ctx;
    load_aux<Sys, R>(ctx, P, node);
    // manufactured forcing while the gather is in flight: after the row/node split it is ~250 instructions on
    // ~40 registers, independent of the populations
    R smms[M];
    if constexpr (MMS) {
        if (staged) {
            if constexpr (PARK > 0) cp_async_wait_1();          // the coefficient group only; the parked populations stay in flight
            else cp_async_wait_all();
            __syncthreads();
            mms_node<Sys, R, true>(P, p, coef_s, smms);
        } else {
            mms_node<Sys, R, false>(P, p, coef, smms);
        }
    }
    if constexpr (PARK > 0) cp_async_wait_all();       // a thread reads only the slots it copied itself: no block barrier
    collide_core<Sys, R, MMS, TRT, PARK, BLOCK>(f, ctx, P, smms, PARK > 0 ? park_s + threadIdx.x : nullptr, [&](auto K, const R* fk) {
        constexpr int k = decltype(K)::value;
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            if constexpr (MODE == MODE_PULL2 || MODE == MODE_LOCAL) {
                dp[(k * Q + i) * TILE] = fk[i];
                if constexpr (PEER) {
                    if (i == 2 * D && plo) plo[(k * Q + i) * TILE] = fk[i];          // slot(-s) -> lower neighbour's upper ghost
                    if (i == 2 * D - 1 && phi) phi[(k * Q + i) * TILE] = fk[i];      // slot(+s) -> upper neighbour's lower ghost
                }
            } else if constexpr (MODE == MODE_AA_EVEN) {
                dp[(k * Q + opposite(i)) * TILE] = fk[i];
            } else {   // AA odd: push to x + c_i; sp[opp(i)] - src + dst is that node (pull source of the opposite direction)
                (dst + (sp[opposite(i)] - src))[(k * Q + i) * TILE] = fk[i];
            }
        }
    });
}

template <class Sys, class R, int MODE, bool MMS, int BLOCK, int MINB, bool TRT = false, bool PEER = false>
__global__ void __launch_bounds__(BLOCK, MINB)
collide_stream_node(typename StepPtr<R, MODE>::Src src, typename StepPtr<R, MODE>::Dst dst, const __grid_constant__ KParams<R> P) {
    constexpr int NCs = MMS ? MmsNC<Sys>::value : 4;
    __shared__ __align__(16) R coef_s[NCs];
    constexpr int PARK = (MMS && !TRT && !PEER && sizeof(R) == 4 && (MODE == MODE_PULL2 || MODE == MODE_LOCAL)) ? ParkCount<Sys>::value : 0;
    __shared__ R park_s[PARK > 0 ? PARK * (2 * Sys::D + 1) * BLOCK : 1];
    node_step<Sys, R, MODE, MMS, BLOCK, false, TRT, PEER, PARK>(src, dst, P, P.coef, P.node0 + (long long)blockIdx.x * BLOCK, coef_s, park_s);
}

// ------------------------------------------------------------------------------------------------ step, persistent
// Launch-free stepping for grids whose state lives in L2 (SURVEY.md §7 "Small configs"): ONE cooperative launch
// advances `nsteps` steps of the two-lattice pull pattern; all blocks are co-resident.  Block b owns the CONTIGUOUS
// node range [b*rounds*BLOCK, (b+1)*rounds*BLOCK) in every step, so what it reads in step s+1 was written in step s by
// the blocks whose ranges lie within one stencil reach (nx nodes in 2D, nx*ny in 3D, cyclically) of its own -- a cyclic
// run of `ndep` blocks starting at `dep0`.  Steps are therefore separated by POINT-TO-POINT flags, not by a grid-wide
// barrier: a block publishes "step s done" in flag[b] and waits only for the flags of its dependency run; the same
// condition covers the write-after-read hazard of the two buffers (a block overwrites in step s+1 what its neighbours
// read in step s).  No global drain: neighbouring blocks may be one step apart.  Step s reads its forcing coefficients
// at P.coef + s*coef_stride.  The per-node code is node_step, i.e. bit-identical to the per-launch path.
// One flag per 128-byte line (FLAG_STRIDE words apart): with 32 flags in a line the pollers of 32 blocks queue at one L2
// sector in front of the stores they wait for (measured on c2: 11.0 us per step packed, 7.8 us one per line).
__device__ __forceinline__ void flags_publish(unsigned int* flag, unsigned int value) {
    // after the block-wide barrier one thread publishes the block's stores with a gpu-scope RELEASE store (cumulative over
    // what the other threads wrote before bar.sync)
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(flag), "r"(value) : "memory");
}
__device__ __forceinline__ void flags_wait(const unsigned int* flags, int dep0, int ndep, int nblocks, unsigned int target) {
    // the first warp polls the dependency run, one flag per lane, with gpu-scope ACQUIRE loads; the populations are then
    // read with ld.global.cg (L2), so no stale L1 line can be observed
    if (threadIdx.x < 32) {
        for (int j = (int)threadIdx.x; j < ndep; j += 32) {
            int d = dep0 + j;
            if (d >= nblocks) d -= nblocks;
            unsigned int v;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(flags + (size_t)d * FLAG_STRIDE) : "memory");
            } while (v < target);
        }
    }
    __syncthreads();
}

// The blocks owning the nodes [first - reach, last + reach] (cyclic): a cyclic run of `ndep` blocks starting at `dep0`
// (every block owns `npb` consecutive nodes, the last one fewer).
__device__ __forceinline__ void dependency_run(long long first, long long last, long long reach, long long npb, long long n, int& dep0, int& ndep) {
    dep0 = 0; ndep = (int)gridDim.x;
    if (last - first + 1 + 2 * reach < n) {
        long long lo = first - reach, hi = last + reach;
        if (lo < 0) lo += n;
        if (hi >= n) hi -= n;
        dep0 = (int)(lo / npb);
        const int dep1 = (int)(hi / npb);
        ndep = (lo > hi && dep0 == dep1) ? (int)gridDim.x : (dep1 - dep0 + (int)gridDim.x) % (int)gridDim.x + 1;
    }
}

template <class Sys, class R, bool MMS, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
collide_stream_persistent(R* fa, R* fb, const __grid_constant__ KParams<R> P, int nsteps, int first_local, long long coef_stride,
                          unsigned int* flags, int rounds) {
    constexpr int NCs = MMS ? MmsNC<Sys>::value : 4;
    __shared__ __align__(16) R coef_s[NCs];
    const long long nseg = (P.n + BLOCK - 1) / BLOCK;
    const bool staged = MMS && NCs >= STAGE_MIN_NC && (P.nx % BLOCK == 0);
    const long long seg0 = (long long)blockIdx.x * rounds, seg1 = seg0 + rounds < nseg ? seg0 + rounds : nseg;
    const long long first = seg0 * BLOCK, last = (seg1 * BLOCK < P.n ? seg1 * BLOCK : P.n) - 1;
    int dep0, ndep;
    dependency_run(first, last, Sys::D == 3 ? (long long)P.nx * P.ny : (long long)P.nx, (long long)rounds * BLOCK, P.n, dep0, ndep);
    R* src = fa;
    R* dst = fb;
    const R* coef = P.coef;
    for (int s = 0; s < nsteps; ++s) {
        for (long long seg = seg0; seg < seg1; ++seg) {
            if (s == 0 && first_local) node_step<Sys, R, MODE_LOCAL, MMS, BLOCK, true>(src, dst, P, coef, seg * BLOCK, coef_s);
            else node_step<Sys, R, MODE_PULL2, MMS, BLOCK, true>(src, dst, P, coef, seg * BLOCK, coef_s);
            if (staged) __syncthreads();          // coef_s is overwritten by the next segment
        }
        R* t = src; src = dst; dst = t;
        coef += coef_stride;
        if (s + 1 < nsteps) {
            flags_publish(flags + (size_t)blockIdx.x * FLAG_STRIDE, (unsigned)(s + 1));
            flags_wait(flags, dep0, ndep, (int)gridDim.x, (unsigned)(s + 1));
        }
    }
}


// The same stepping with FAT blocks: GROUPS x BLOCK threads, one block per SM, each group of BLOCK threads takes whole segments.
// A block then owns enough rows to have an INTERIOR (segments further than one stencil reach from both ends of its range, which
// touch no other block's nodes): per step it waits for its neighbours' flags, updates its boundary segments, publishes its own
// flag and only then updates the interior -- the flag's round trip through L2 is hidden behind the interior work.  flag[b] = s+1
// now means "block b has finished the BOUNDARY segments of step s", which is all its neighbours depend on (they read and, one
// step later, their reads of b's nodes are what b's next writes must not overtake: both happen in their boundary phase).
// Only without shared-memory staging of the row coefficients (node_step's staging is per block); same node_step, same bits.
template <class Sys, class R, bool MMS, int BLOCK, int GROUPS>
__global__ void __launch_bounds__(BLOCK * GROUPS, 1)
collide_stream_persistent_fat(R* fa, R* fb, const __grid_constant__ KParams<R> P, int nsteps, int first_local, long long coef_stride,
                              unsigned int* flags, int rounds) {
    static_assert(!(MMS && MmsNC<Sys>::value >= STAGE_MIN_NC), "fat blocks: unstaged row coefficients only");
    const long long nseg = (P.n + BLOCK - 1) / BLOCK;
    const long long seg0 = (long long)blockIdx.x * rounds, seg1 = seg0 + rounds < nseg ? seg0 + rounds : nseg;
    const long long first = seg0 * BLOCK, last = (seg1 * BLOCK < P.n ? seg1 * BLOCK : P.n) - 1;
    const long long reach = Sys::D == 3 ? (long long)P.nx * P.ny : (long long)P.nx;
    int dep0, ndep;
    dependency_run(first, last, reach, (long long)rounds * BLOCK, P.n, dep0, ndep);
    // interior segments [sb0, sb1): every node in [first + reach, last - reach]
    long long sb0 = (first + reach + BLOCK - 1) / BLOCK, sb1 = (last - reach + 1) / BLOCK;
    if (sb0 > seg1) sb0 = seg1;
    if (last - reach + 1 < first || sb1 < sb0) sb1 = sb0;
    if (gridDim.x == 1) { sb0 = seg0; sb1 = seg1; }                      // a single block has no boundary
    const long long nlo = sb0 - seg0, nbd = nlo + (seg1 - sb1);
    const int grp = (int)threadIdx.x / BLOCK;
    const long long goff = (long long)grp * BLOCK;                          // node_step adds threadIdx.x to `first`
    R* src = fa;
    R* dst = fb;
    const R* coef = P.coef;
    for (int s = 0; s < nsteps; ++s) {
        if (s > 0) flags_wait(flags, dep0, ndep, (int)gridDim.x, (unsigned)s);
        const bool local = s == 0 && first_local;
        for (long long j = grp; j < nbd; j += GROUPS) {
            const long long seg = j < nlo ? seg0 + j : sb1 + (j - nlo);
            if (local) node_step<Sys, R, MODE_LOCAL, MMS, BLOCK, true>(src, dst, P, coef, seg * BLOCK - goff, nullptr);
            else node_step<Sys, R, MODE_PULL2, MMS, BLOCK, true>(src, dst, P, coef, seg * BLOCK - goff, nullptr);
        }
        if (s + 1 < nsteps) flags_publish(flags + (size_t)blockIdx.x * FLAG_STRIDE, (unsigned)(s + 1));
        for (long long seg = sb0 + grp; seg < sb1; seg += GROUPS) {
            if (local) node_step<Sys, R, MODE_LOCAL, MMS, BLOCK, true>(src, dst, P, coef, seg * BLOCK - goff, nullptr);
            else node_step<Sys, R, MODE_PULL2, MMS, BLOCK, true>(src, dst, P, coef, seg * BLOCK - goff, nullptr);
        }
        R* t = src; src = dst; dst = t;
        coef += coef_stride;
    }
}

// ------------------------------------------------------------------------------------------------ step, SM-resident
// Grids whose ONE population copy fits in the shared memory of the whole GPU (148 x 227 KB = 33 MB; c2 in fp64 is 31 MB):
// one cooperative launch, one block per SM; block b owns a contiguous run of tiles and keeps them in shared memory IN THE
// GLOBAL LAYOUT (shared element = global element - shift), stepped in place with the AA pattern (even step: a node reads and
// rewrites its own slots, swapped; odd step: it reads slot opp(i) of x - c_i and writes slot i of x + c_i -- the same slot set,
// so no staging and no second copy).  Slot (x, s) is touched by node x on even and by node x - c_s on odd steps: when both
// belong to the block it lives in shared memory, otherwise it STAYS IN GLOBAL MEMORY (L2) and both blocks access it there --
// the block-boundary populations are the only per-step traffic that leaves the SM.  Steps are separated by the same
// point-to-point flags as in collide_stream_persistent (every global-homed slot is written in one step by one block and read
// in the next by the other).  Pointers are generic (shared or global), the arithmetic is collide_core.  Entry: the tiles are
// copied in; exit: the shared-homed slots are copied back (the global-homed ones are already in place).
template <class Sys, class R, bool ODD, bool MMS>
__device__ __forceinline__ void node_step_generic(R* const (&sp)[2 * Sys::D + 1], const KParams<R>& P, const R* coef, long long node, const NodeIdx& p) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    R f[M][Q];
#pragma unroll
    for (int k = 0; k < M; ++k)
#pragma unroll
        for (int i = 0; i < Q; ++i) f[k][i] = sp[i][(k * Q + (ODD ? opposite(i) : i)) * TILE];
    typename Sys::Ctx ctx;
    load_aux<Sys, R>(ctx, P, node);
    R smms[M];
    if constexpr (MMS) mms_node<Sys, R, false>(P, p, coef, smms);
    collide_core<Sys, R, MMS>(f, ctx, P, smms, nullptr, [&](auto K, const R* fk) {
        constexpr int k = decltype(K)::value;
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            if constexpr (ODD) sp[opposite(i)][(k * Q + i) * TILE] = fk[i];                  // slot i of x + c_i (the pull source of opp(i))
            else sp[opposite(i)][(k * Q + opposite(i)) * TILE] = fk[i];                      // own slot opp(i)
        }
    });
}

template <class Sys, class R, bool MMS, int BLOCK>
__global__ void __launch_bounds__(BLOCK, 1)
collide_stream_resident(R* f, const __grid_constant__ KParams<R> P, int nsteps, int parity0, long long coef_stride, unsigned int* flags, int rounds) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M, MQ = M * Q, G = BLOCK / TILE;
    static_assert(BLOCK % TILE == 0, "whole tiles per pass");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    R* const sm = reinterpret_cast<R*>(smem_raw);
    const long long ntile = (P.n + TILE - 1) / TILE;
    const long long t0 = (long long)blockIdx.x * rounds, t1 = t0 + rounds < ntile ? t0 + rounds : ntile;
    const long long first = t0 * TILE, last = (t1 * TILE < P.n ? t1 * TILE : P.n) - 1;
    const long long shift = t0 * (long long)MQ * TILE;
    int dep0, ndep;
    dependency_run(first, last, D == 3 ? (long long)P.nx * P.ny : (long long)P.nx, (long long)rounds * TILE, P.n, dep0, ndep);
    {
        const long long own = (t1 - t0) * (long long)MQ * TILE;
        for (long long e = threadIdx.x; e < own; e += BLOCK) sm[e] = f[shift + e];
    }
    __syncthreads();
    const int lane = (int)threadIdx.x & (TILE - 1), grp = (int)threadIdx.x >> LOG_TILE;
    // boundary tiles (some node has a neighbour outside the block: within one reach of either end) go first in every step, then
    // the flag is published, then the interior tiles (shared memory only) run while the flag travels to the neighbours
    const long long reach = D == 3 ? (long long)P.nx * P.ny : (long long)P.nx;
    long long tb0 = (first + reach - 1) / TILE + 1, tb1 = (last - reach + 1) / TILE;
    if (tb0 > t1) tb0 = t1;
    if (last - reach + 1 < first || tb1 < tb0) tb1 = tb0;
    if (dep0 == 0 && ndep == (int)gridDim.x && gridDim.x == 1) { tb0 = t0; tb1 = t1; }        // a single block has no boundary
    const long long nlo = tb0 - t0, nbd = nlo + (t1 - tb1);
    auto tile_step = [&](long long t, bool odd, const R* coef) {
        const long long node = t * TILE + lane;
        if (node < P.n) {
            const NodeIdx p = decompose(node, P.nx, P.ny);
            R* sp[Q];
#pragma unroll
            for (int i = 0; i < Q; ++i) {
                const long long sn = node + pull_offset(i, p, P.nx, P.ny, P.nz);
                const long long off = tile_off(odd ? sn : node, MQ);
                sp[i] = (sn >= first && sn <= last) ? sm + (off - shift) : f + off;
            }
            if (odd) node_step_generic<Sys, R, true, MMS>(sp, P, coef, node, p);
            else node_step_generic<Sys, R, false, MMS>(sp, P, coef, node, p);
        }
    };
    const R* coef = P.coef;
    for (int s = 0; s < nsteps; ++s) {
        const bool odd = ((parity0 + s) & 1) != 0;
        if (s > 0) flags_wait(flags, dep0, ndep, (int)gridDim.x, (unsigned)s);      // the neighbours' boundary tiles of step s-1 are done
        for (long long j = grp; j < nbd; j += G) tile_step(j < nlo ? t0 + j : tb1 + (j - nlo), odd, coef);
        if (s + 1 < nsteps) flags_publish(flags + (size_t)blockIdx.x * FLAG_STRIDE, (unsigned)(s + 1));
        for (long long t = tb0 + grp; t < tb1; t += G) tile_step(t, odd, coef);
        coef += coef_stride;
    }
    __syncthreads();
    for (long long t = t0 + grp; t < t1; t += G) {
        const long long node = t * TILE + lane;
        if (node < P.n) {
            const NodeIdx p = decompose(node, P.nx, P.ny);
            const long long off = tile_off(node, MQ);
#pragma unroll
            for (int i = 0; i < Q; ++i) {
                const long long sn = node + pull_offset(i, p, P.nx, P.ny, P.nz);
                if (sn >= first && sn <= last) {
#pragma unroll
                    for (int k = 0; k < M; ++k) f[off + (k * Q + i) * TILE] = sm[off - shift + (k * Q + i) * TILE];
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ step, cluster-resident
// Grids of a few thousand nodes (configs[0]: 64 x 64) do not even fill L2 lines worth a barrier through L2: ONE thread-block
// cluster of up to 8 CTAs holds the whole population state in DISTRIBUTED SHARED MEMORY, one node per thread.  Step 0 gathers
// from global memory (as the per-launch kernel would), the steps between go shared -> shared through two buffers per CTA -- a
// pull across a CTA boundary is a DSMEM load from the owner CTA's buffer -- with one hardware cluster barrier per step, and the
// last step stores to global memory in the usual post-collision form.  Arithmetic: collide_core, i.e. the same bits.
// smem per CTA: R[2][M*Q][npc] (npc = nodes per CTA = blockDim.x).  No forcing, no prescribed fields (small tracker-free
// systems); everything else falls back to collide_stream_persistent.
template <class Sys, class R>
__global__ void __launch_bounds__(1024, 1)
collide_stream_cluster(const R* __restrict__ gsrc, R* __restrict__ gdst, const __grid_constant__ KParams<R> P, int nsteps, int first_local) {
    namespace cg = cooperative_groups;
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    R* const sm = reinterpret_cast<R*>(smem_raw);
    const int npc = (int)blockDim.x;
    const int rank = (int)cluster.block_rank();
    const long long node = (long long)rank * npc + threadIdx.x;
    const bool active = node < P.n;
    const long long bufsz = (long long)M * Q * npc;
    // where this node pulls direction i from, in buffer 0 of the owner CTA (buffer 1: + bufsz); fixed for the whole launch
    const R* sp0[Q];
    long long goff[Q];
    NodeIdx p = {0, 0, 0};
    if (active) {
        p = decompose(node, P.nx, P.ny);
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            const long long sn = node + pull_offset(i, p, P.nx, P.ny, P.nz);
            const int owner = (int)(sn / npc), loc = (int)(sn - (long long)owner * npc);
            const R* base = owner == rank ? sm : cluster.map_shared_rank(sm, owner);
            sp0[i] = base + (long long)i * npc + loc;                     // + k*Q*npc per component
            goff[i] = tile_off(first_local ? node : sn, M * Q);
        }
    }
    cluster.sync();                                                       // every CTA of the cluster is resident before any DSMEM access
    R smms[M];
    for (int s = 0; s < nsteps; ++s) {
        if (active) {
            R f[M][Q];
            const long long rd = ((s - 1) & 1) * bufsz;                   // step s >= 1 reads what step s-1 wrote
#pragma unroll
            for (int k = 0; k < M; ++k)
#pragma unroll
                for (int i = 0; i < Q; ++i)
                    f[k][i] = s == 0 ? gsrc[goff[i] + (k * Q + i) * TILE] : sp0[i][rd + (long long)(k * Q) * npc];
            typename Sys::Ctx ctx;
            const bool last = s == nsteps - 1;
            R* const wr = sm + (s & 1) * bufsz + threadIdx.x;
            R* const gp = gdst + tile_off(node, M * Q);
            collide_core<Sys, R, false>(f, ctx, P, smms, nullptr, [&](auto K, const R* fk) {
                constexpr int k = decltype(K)::value;
#pragma unroll
                for (int i = 0; i < Q; ++i) {
                    if (last) gp[(k * Q + i) * TILE] = fk[i];
                    else wr[(long long)(k * Q + i) * npc] = fk[i];
                }
            });
        }
        cluster.sync();                  // release/acquire at cluster scope: the shared-memory stores are visible to the DSMEM loads
    }
}

// ------------------------------------------------------------------------------------------------ step, several nodes per thread
// Single-field systems (Burgers, advection: 5 populations per node) do not keep enough loads in flight with one node per
// thread to cover the HBM latency (64 warps x 5 loads x 128 B = 41 KB per SM against ~37 KB needed by Little's law: 94 % of the
// copy peak).  Here a thread gathers NPT nodes (BLOCK apart, so every warp access stays one full 128-byte line) before it
// collides any of them: NPT x the memory-level parallelism, same collide_core.  Two-lattice modes, no forcing, no prescribed fields.
template <class Sys, class R, int MODE, int BLOCK, int NPT>
__global__ void __launch_bounds__(BLOCK)
collide_stream_multi(typename StepPtr<R, MODE>::Src src, typename StepPtr<R, MODE>::Dst dst, const __grid_constant__ KParams<R> P) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    static_assert(MODE == MODE_PULL2 || MODE == MODE_LOCAL, "two-lattice modes only");
    const long long first = P.node0 + (long long)blockIdx.x * (BLOCK * NPT) + threadIdx.x;
    R f[NPT][M][Q];
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        const long long node = first + (long long)j * BLOCK;
        if (node < P.node1) {
            const NodeIdx p = decompose(node, P.nx, P.ny);
#pragma unroll
            for (int i = 0; i < Q; ++i) {
                const R* sp = src + tile_off(node + (MODE == MODE_LOCAL ? 0LL : pull_offset(i, p, P.nx, P.ny, P.nz)), M * Q);
#pragma unroll
                for (int k = 0; k < M; ++k) f[j][k][i] = sp[(k * Q + i) * TILE];
            }
        }
    }
    R smms[M];
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        const long long node = first + (long long)j * BLOCK;
        if (node < P.node1) {
            typename Sys::Ctx ctx;
            R* const dp = dst + tile_off(node, M * Q);
            collide_core<Sys, R, false>(f[j], ctx, P, smms, nullptr, [&](auto K, const R* fk) {
                constexpr int k = decltype(K)::value;
#pragma unroll
                for (int i = 0; i < Q; ++i) dp[(k * Q + i) * TILE] = fk[i];
            });
        }
    }
}

// ------------------------------------------------------------------------------------------------ step, two-pass
// Low-register variant using the linearity of BGK in f (SURVEY.md §7 option iii):
//   f'_k,i = (1 - omega_k) f_k,i + c_k,i,   c_k,0 = w0 (omega dQ_k + s_k),  c_k,+-a = w1 (omega dQ_k + s_k) +- (omega/2) dF_k,a.
// Pass 1 streams the Q*M populations through one register each and keeps only the M moments; pass 2 reads
// them again (L1/L2 hits: the same thread touched the same sectors microseconds earlier; DRAM traffic is
// unchanged) and writes f'.  ~3x fewer live registers than the node kernel -> 2-3x the resident warps.
template <class Sys, class R, int MODE, bool MMS, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
collide_stream_twopass(typename StepPtr<R, MODE>::Src src, typename StepPtr<R, MODE>::Dst dst, const __grid_constant__ KParams<R> P) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    using L = Lattice<D>;
    const long long node = P.node0 + (long long)blockIdx.x * BLOCK + threadIdx.x;
    if (node >= P.node1) return;
    const NodeIdx p = decompose(node, P.nx, P.ny);
    R smms[M];
    if constexpr (MMS) mms_node<Sys, R, false>(P, p, P.coef, smms);
    const R* sp[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i)
        sp[i] = src + tile_off(node + ((MODE == MODE_AA_EVEN || MODE == MODE_LOCAL) ? 0LL : pull_offset(i, p, P.nx, P.ny, P.nz)), M * Q);
    R* const dp = dst + tile_off(node, M * Q);
    R dQ[M];
#pragma unroll
    for (int k = 0; k < M; ++k) {
        R s = R(0);
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            const int slot = (MODE == MODE_AA_ODD) ? opposite(i) : i;
            const R v = sp[i][(k * Q + slot) * TILE];
            s = (i == 0) ? v : s + v;                     // same summation order as the node kernel
        }
        dQ[k] = s;
    }
    typename Sys::Ctx ctx;
    load_aux<Sys, R>(ctx, P, node);
    Sys::setup(ctx, dQ, P);
    static_for<0, M>([&](auto K) {
        constexpr int k = decltype(K)::value;
        R F[D], S;
        Sys::template flux<k>(ctx, dQ, P, F, S);
        if constexpr (MMS) S += smms[k];
        R f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            const int slot = (MODE == MODE_AA_ODD) ? opposite(i) : i;
            f[i] = sp[i][(k * Q + slot) * TILE];
        }
        relax<D, R>(f, P.omega[k], dQ[k], F, S);
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            if constexpr (MODE == MODE_PULL2 || MODE == MODE_LOCAL) {
                dp[(k * Q + i) * TILE] = f[i];
            } else if constexpr (MODE == MODE_AA_EVEN) {
                dp[(k * Q + opposite(i)) * TILE] = f[i];
            } else {
                (dst + (sp[opposite(i)] - src))[(k * Q + i) * TILE] = f[i];
            }
        }
    });
}

// ------------------------------------------------------------------------------------------------ init
// step 0: f*_k,i = w_i (dQ_k + c_i . dF_k / c_s^2),  dQ = U - Q0 (subtracted in fp64), eq 2.23
template <class Sys, class R>
__global__ void init_from_U_kernel(const double* __restrict__ U, long long ustride, long long node0, long long node1, R* __restrict__ f,
                                   const __grid_constant__ KParams<R> P, const __grid_constant__ KParams<double> Pd) {
    // nodes [node0, node1); U holds that node range, component planes `ustride` apart (the whole grid: 0, n, n)
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    const long long node = node0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= node1) return;
    R dQ[M];
#pragma unroll
    for (int k = 0; k < M; ++k) dQ[k] = (R)(U[(long long)k * ustride + (node - node0)] - Pd.ref[k]);
    typename Sys::Ctx ctx;
    load_aux<Sys, R>(ctx, P, node);
    Sys::setup(ctx, dQ, P);
    static_for<0, M>([&](auto K) {
        constexpr int k = decltype(K)::value;
        R F[D], S;
        Sys::template flux<k>(ctx, dQ, P, F, S);
        using L = Lattice<D>;
        f[tile_off(node, M * Q) + (k * Q) * TILE] = weight0<D, R>() * dQ[k];
#pragma unroll
        for (int a = 0; a < D; ++a) {
            const R h = R(0.5) * F[a];              // w1 / c_s^2 = 1/2
            f[tile_off(node, M * Q) + (k * Q + 1 + 2 * a) * TILE] = R(L::w1) * dQ[k] + h;
            f[tile_off(node, M * Q) + (k * Q + 2 + 2 * a) * TILE] = R(L::w1) * dQ[k] - h;
        }
    });
}

// Equilibrium of the reference state in fp64, feq0[k*Q+i] = w_i (Q0_k + c_i.F_k(Q0)/c_s^2): what the shifted
// storage subtracts (eq 2.23).  One thread; runs once per grid.
template <class Sys>
__global__ void reference_equilibrium_kernel(double* __restrict__ feq0, const __grid_constant__ KParams<double> P0 /*ref = 0*/,
                                             const __grid_constant__ KParams<double> Pd) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    double Q0[M];
    bool any = false;
    for (int k = 0; k < M; ++k) { Q0[k] = Pd.ref[k]; any = any || (Q0[k] != 0.0); }
    if (!any) { for (int q = 0; q < M * Q; ++q) feq0[q] = 0.0; return; }
    typename Sys::Ctx ctx;
    if constexpr (AuxCount<Sys>::value > 0) Sys::default_aux(ctx);     // uniform reference: the prescribed fields drop out
    Sys::setup(ctx, Q0, P0);
    static_for<0, M>([&](auto K) {
        constexpr int k = decltype(K)::value;
        double F[D], S;
        Sys::template flux<k>(ctx, Q0, P0, F, S);
        using L = Lattice<D>;
        feq0[k * Q] = L::w0 * Q0[k];
        for (int a = 0; a < D; ++a) {
            feq0[k * Q + 1 + 2 * a] = L::w1 * (Q0[k] + F[a] / L::cs2);
            feq0[k * Q + 2 + 2 * a] = L::w1 * (Q0[k] - F[a] / L::cs2);
        }
    });
}

// ------------------------------------------------------------------------------------------------ readback
// canonical gather: population (k, i) of `node` sits in slot i at node (GATHER_CANON), in slot opp(i) at
// node - c_i (GATHER_AA_ODD) or in slot i at node - c_i (GATHER_PULL).
template <int Q, class R>
__device__ __forceinline__ R load_canonical(const R* __restrict__ f, int M, int k, int i, long long node,
                                            const NodeIdx& p, int nx, int ny, int nz, int gather) {
    if (gather == GATHER_CANON) return f[tile_off(node, M * Q) + (k * Q + i) * TILE];
    const int slot = gather == GATHER_AA_ODD ? opposite(i) : i;
    return f[tile_off(node + pull_offset(i, p, nx, ny, nz), M * Q) + (k * Q + slot) * TILE];
}

// U_k = Q0_k + sum_i f*_k,i, accumulated and returned in fp64 (eq 2.6; reading A17)
template <int Q, class R>
__global__ void read_U_kernel(const R* __restrict__ f, double* __restrict__ U, long long ustride, long long node0, long long node1, int M,
                              int nx, int ny, int nz, int gather, const __grid_constant__ KParams<double> Pd) {
    // nodes [node0, node1) into U, component planes `ustride` apart (the whole grid: n, 0, n)
    const long long node = node0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= node1) return;
    const NodeIdx p = decompose(node, nx, ny);
    for (int k = 0; k < M; ++k) {
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < Q; ++i) s += (double)load_canonical<Q, R>(f, M, k, i, node, p, nx, ny, nz, gather);
        U[(long long)k * ustride + (node - node0)] = Pd.ref[k] + s;
    }
}

template <int Q, class R>
__global__ void read_f_kernel(const R* __restrict__ f, double* __restrict__ out, const double* __restrict__ feq0, int M,
                              int nx, int ny, int nz, long long n, int gather) {
    const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= n) return;
    const NodeIdx p = decompose(node, nx, ny);
    for (int k = 0; k < M; ++k)
#pragma unroll
        for (int i = 0; i < Q; ++i)
            out[(long long)(k * Q + i) * n + node] =
                (double)load_canonical<Q, R>(f, M, k, i, node, p, nx, ny, nz, gather) + feq0[k * Q + i];
}

template <class R>
__global__ void set_f_kernel(const double* __restrict__ in, R* __restrict__ f, const double* __restrict__ feq0, int MQ, long long n) {   // in: [plane][node]
    const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= n) return;
    for (int q = 0; q < MQ; ++q) f[tile_off(node, MQ) + q * TILE] = (R)(in[(long long)q * n + node] - feq0[q]);
}

// prescribed coefficient fields: user fp64 [NA][n] -> R [NA][aux_stride]
template <class R>
__global__ void set_aux_kernel(const double* __restrict__ in, R* __restrict__ aux, int NA, long long n, long long stride) {
    const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= n) return;
    for (int a = 0; a < NA; ++a) aux[a * stride + node] = (R)in[(long long)a * n + node];
}

// ghost plane of a slab: first / last plane of the slowest axis
template <int D> __device__ __forceinline__ bool is_ghost(const NodeIdx& p, int ny, int nz) {
    return D == 3 ? (p.iz == 0 || p.iz == nz - 1) : (p.iy == 0 || p.iy == ny - 1);
}

// ------------------------------------------------------------------------------------------------ a10
// Sub-characteristic check (eq 2.19-2.20; L329): max over nodes of the system's wave
// speeds, in fp64 from the canonical moments.  Warp shuffle -> shared -> one atomicMax per block on the
// bit pattern (non-negative doubles order like unsigned integers).  out3 must be zeroed before launch.
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
// max that does not lose a blown-up state: fmax() returns the non-NaN operand, so a NaN candidate is turned into +inf
// (which the shuffle / atomicMax-on-the-bit-pattern reductions then carry to the host, where it fails `<= c_s`).
__device__ __forceinline__ double max_nan_inf(double m, double v) { return (v == v) ? fmax(m, v) : (double)INFINITY; }

template <class Sys, class R>
__global__ void __launch_bounds__(256)
max_wave_speed_kernel(const R* __restrict__ f, unsigned long long* __restrict__ out3, long long n, int nx, int ny, int nz,
                      int gather, const __grid_constant__ KParams<double> Pd) {
    constexpr int Q = 2 * Sys::D + 1, M = Sys::M;
    double m[3] = {0.0, 0.0, 0.0};
    for (long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x; node < n; node += (long long)gridDim.x * blockDim.x) {
        const NodeIdx p = decompose(node, nx, ny);
        if (Pd.ghost && is_ghost<Sys::D>(p, ny, nz)) continue;
        double U[M], w[3];
        for (int k = 0; k < M; ++k) {
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < Q; ++i) s += (double)load_canonical<Q, R>(f, M, k, i, node, p, nx, ny, nz, gather);
            U[k] = Pd.ref[k] + s;
        }
        Sys::wave(U, Pd, w);
        m[0] = max_nan_inf(m[0], w[0] * Pd.il);     // physical speed / lambda
        m[1] = max_nan_inf(m[1], w[1] * Pd.il);
        m[2] = max_nan_inf(m[2], w[2]);             // already lattice
    }
    __shared__ double sm[3][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const double v = warp_max(m[j]);
        if (lane == 0) sm[j][warp] = v;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            double v = lane < (int)(blockDim.x >> 5) ? sm[j][lane] : 0.0;
            v = warp_max(v);
            if (lane == 0) atomicMax(out3 + j, (unsigned long long)__double_as_longlong(v));
        }
    }
}

// ------------------------------------------------------------------------------------------------ error norms
// Convergence-study reductions: per component k the sums that make the relative L1, L2 and
// Linf errors of the current state against the manufactured solution at the current time,
//   out[k] = { sum|e|, sum e^2, max|e|, sum|q|, sum q^2, max|q| },  e = U_k - Q_exact,k,  q = Q_exact,k,
// everything in fp64: the exact state is evaluated from the closed forms (no tables), U_k from the canonical
// populations.  Warp shuffle -> shared -> one atomic per block and quantity.  out must be zeroed before launch.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <class Sys, class R>
__global__ void __launch_bounds__(256)
error_norms_kernel(const R* __restrict__ f, double* __restrict__ out, long long n, int nx, int ny, int nz, int gather, double t,
                   const __grid_constant__ MmsHostArgs mh, const __grid_constant__ KParams<double> Pd) {
    if constexpr (has_mms<Sys>()) {
        constexpr int Q = 2 * Sys::D + 1, M = Sys::M;
        using G = typename Sys::Mms;
        double acc[M][6];
        for (int k = 0; k < M; ++k) for (int j = 0; j < 6; ++j) acc[k][j] = 0.0;
        double T[8];
        G::time_scalars(t, mh, T);
        for (long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x; node < n; node += (long long)gridDim.x * blockDim.x) {
            const NodeIdx p = decompose(node, nx, ny);
            double X[8], Y[8], Z[8], q[M];
            if (Pd.ghost && is_ghost<Sys::D>(p, ny, nz)) continue;
            G::axis_row(0, (p.ix + Pd.ox) * mh.dx, mh, X);
            G::axis_row(1, (p.iy + Pd.oy) * mh.dx, mh, Y);
            if (G::NZ > 0) G::axis_row(2, (p.iz + Pd.oz) * mh.dx, mh, Z);
            G::template exact<double>(Pd.mms, T, X, Y, Z, q);
            for (int k = 0; k < M; ++k) {
                double s = 0.0;
#pragma unroll
                for (int i = 0; i < Q; ++i) s += (double)load_canonical<Q, R>(f, M, k, i, node, p, nx, ny, nz, gather);
                const double e = fabs(Pd.ref[k] + s - q[k]), a = fabs(q[k]);
                acc[k][0] += e; acc[k][1] += e * e; acc[k][2] = max_nan_inf(acc[k][2], e);
                acc[k][3] += a; acc[k][4] += a * a; acc[k][5] = max_nan_inf(acc[k][5], a);
            }
        }
        __shared__ double sm[8];
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        for (int k = 0; k < M; ++k)
            for (int j = 0; j < 6; ++j) {
                const bool is_max = (j == 2 || j == 5);
                double v = is_max ? warp_max(acc[k][j]) : warp_sum(acc[k][j]);
                if (lane == 0) sm[warp] = v;
                __syncthreads();
                if (warp == 0) {
                    v = lane < (int)(blockDim.x >> 5) ? sm[lane] : 0.0;
                    v = is_max ? warp_max(v) : warp_sum(v);
                    if (lane == 0) {
                        if (is_max) atomicMax(reinterpret_cast<unsigned long long*>(out + k * 6 + j), (unsigned long long)__double_as_longlong(v));
                        else atomicAdd(out + k * 6 + j, v);
                    }
                }
                __syncthreads();
            }
    }
}

// ---- the same norms without atomics, through caller-independent scratch (lbmk_error_norms_noalloc): pass 1 writes one RECORD
// [M][6] per NORM_RECORD_NODES consecutive nodes (one block per record, fixed summation tree), pass 2 combines the records in index
// order, so the result does not depend on the SM count or on scheduling.  Every record of [0, nrec) is fully written by pass 1:
// nothing in the scratch has to be cleared.

template <class Sys, class R>
__global__ void __launch_bounds__(256)
error_norm_records_kernel(const R* __restrict__ f, double* __restrict__ rec, long long n, int nx, int ny, int nz, int gather, double t,
                          const __grid_constant__ MmsHostArgs mh, const __grid_constant__ KParams<double> Pd) {
    if constexpr (has_mms<Sys>()) {
        constexpr int Q = 2 * Sys::D + 1, M = Sys::M;
        using G = typename Sys::Mms;
        double acc[M][6];
        for (int k = 0; k < M; ++k) for (int j = 0; j < 6; ++j) acc[k][j] = 0.0;
        double T[8];
        G::time_scalars(t, mh, T);
        const long long first = (long long)blockIdx.x * NORM_RECORD_NODES;
        const long long last = first + NORM_RECORD_NODES < n ? first + NORM_RECORD_NODES : n;
        for (long long node = first + threadIdx.x; node < last; node += blockDim.x) {
            const NodeIdx p = decompose(node, nx, ny);
            double X[8], Y[8], Z[8], q[M];
            if (Pd.ghost && is_ghost<Sys::D>(p, ny, nz)) continue;
            G::axis_row(0, (p.ix + Pd.ox) * mh.dx, mh, X);
            G::axis_row(1, (p.iy + Pd.oy) * mh.dx, mh, Y);
            if (G::NZ > 0) G::axis_row(2, (p.iz + Pd.oz) * mh.dx, mh, Z);
            G::template exact<double>(Pd.mms, T, X, Y, Z, q);
            for (int k = 0; k < M; ++k) {
                double s = 0.0;
#pragma unroll
                for (int i = 0; i < Q; ++i) s += (double)load_canonical<Q, R>(f, M, k, i, node, p, nx, ny, nz, gather);
                const double e = fabs(Pd.ref[k] + s - q[k]), a = fabs(q[k]);
                acc[k][0] += e; acc[k][1] += e * e; acc[k][2] = max_nan_inf(acc[k][2], e);
                acc[k][3] += a; acc[k][4] += a * a; acc[k][5] = max_nan_inf(acc[k][5], a);
            }
        }
        __shared__ double sm[8][M * 6];
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        for (int k = 0; k < M; ++k)
            for (int j = 0; j < 6; ++j) {
                const double v = (j == 2 || j == 5) ? warp_max(acc[k][j]) : warp_sum(acc[k][j]);
                if (lane == 0) sm[warp][k * 6 + j] = v;
            }
        __syncthreads();
        for (int q = threadIdx.x; q < M * 6; q += blockDim.x) {
            const bool is_max = (q % 6 == 2 || q % 6 == 5);
            double v = sm[0][q];
            for (int w = 1; w < 8; ++w) v = is_max ? max_nan_inf(v, sm[w][q]) : v + sm[w][q];
            rec[(long long)blockIdx.x * (M * 6) + q] = v;
        }
    }
}

// pass 2: out[q] = records combined in index order; one thread per (component, quantity)
static __global__ void combine_norm_records_kernel(const double* __restrict__ rec, long long nrec, int MQ6, double* __restrict__ out) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= MQ6) return;
    const bool is_max = (q % 6 == 2 || q % 6 == 5);
    double v = rec[q];
    for (long long r = 1; r < nrec; ++r) {
        const double x = rec[r * MQ6 + q];
        v = is_max ? max_nan_inf(v, x) : v + x;
    }
    out[q] = v;
}

// ------------------------------------------------------------------------------------------------ flux self-check
// Every node of the current state: the hand-written delta form (Sys<double>: dF = F(Q0 + dQ) - F(Q0), s(Q0 + dQ)) against the
// generated plain form (Gen: F(U), s(U); gen/cascade.py), in fp64.  out[0] = max over nodes and components of
// |dF_hand - (F_gen(U) - F_gen(Q0))| and |s_hand - s_gen| relative to the node's largest |F_gen|, |s_gen| entry.
template <class Sys, class Gen, class R>
__global__ void __launch_bounds__(128)
flux_selfcheck_kernel(const R* __restrict__ f, const R* __restrict__ aux, long long aux_stride, unsigned long long* __restrict__ out,
                      long long n, int nx, int ny, int nz, int gather, const __grid_constant__ KParams<double> Pd,
                      const __grid_constant__ GenArgs<double> ga) {
    constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M, NA = AuxCount<Sys>::value;
    double worst = 0.0;
    double F0[M * D], S0[M], Q0[M], A[NA > 0 ? NA : 1];
    for (long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x; node < n; node += (long long)gridDim.x * blockDim.x) {
        const NodeIdx p = decompose(node, nx, ny);
        double U[M], dQ[M];
        for (int k = 0; k < M; ++k) {
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < Q; ++i) s += (double)load_canonical<Q, R>(f, M, k, i, node, p, nx, ny, nz, gather);
            dQ[k] = s; Q0[k] = Pd.ref[k]; U[k] = Pd.ref[k] + s;
        }
        for (int a = 0; a < NA; ++a) A[a] = (double)aux[a * aux_stride + node];
        typename Sys::Ctx ctx;
        if constexpr (NA > 0) { double Aa[NA > 0 ? NA : 1]; for (int a = 0; a < NA; ++a) Aa[a] = A[a]; Sys::set_aux(ctx, Aa); }
        Sys::setup(ctx, dQ, Pd);
        double Fg[M * D], Sg[M];
        Gen::template flux<double>(U, A, ga, Fg, Sg);
        bool shifted = false;
        for (int k = 0; k < M; ++k) shifted = shifted || Q0[k] != 0.0;
        if (shifted) Gen::template flux<double>(Q0, A, ga, F0, S0);
        else for (int q = 0; q < M * D; ++q) F0[q] = 0.0;
        double scale = 1e-300;
        for (int q = 0; q < M * D; ++q) scale = fmax(scale, fabs(Fg[q]));
        for (int k = 0; k < M; ++k) scale = fmax(scale, fabs(Sg[k]));
        static_for<0, M>([&](auto K) {
            constexpr int k = decltype(K)::value;
            double F[D], S;
            Sys::template flux<k>(ctx, dQ, Pd, F, S);
            for (int a = 0; a < D; ++a) worst = max_nan_inf(worst, fabs(F[a] - (Fg[k * D + a] - F0[k * D + a])) / scale);
            worst = max_nan_inf(worst, fabs(S - Sg[k]) / scale);
        });
    }
    worst = warp_max(worst);
    if ((threadIdx.x & 31) == 0) atomicMax(out, (unsigned long long)__double_as_longlong(worst));
}

// ------------------------------------------------------------------------------------------------ a11
// Dirichlet-MMS frame (reading A18; the paper defines no boundary operator):
// the outermost node layer is reset to f_eq(Q_exact(x_b, t_n)) in canonical slots.  One thread per frame
// node candidate; P.T holds the time scalars at t_n (not the midpoint).  Two-lattice storage only: with the
// stream pending (GATHER_PULL) the canonical population (i, x_b) is written where the next pull finds it.
template <class Sys, class R>
__global__ void dirichlet_frame_kernel(R* __restrict__ f, int gather, const __grid_constant__ KParams<R> P, const __grid_constant__ KParams<double> Pd) {
    if constexpr (has_mms<Sys>()) {
        constexpr int D = Sys::D, Q = 2 * D + 1, M = Sys::M;
        using G = typename Sys::Mms;
        const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (node >= P.n) return;
        const NodeIdx p = decompose(node, P.nx, P.ny);
        bool frame = p.ix == 0 || p.ix == P.nx - 1 || p.iy == 0 || p.iy == P.ny - 1;
        if (D == 3) frame = frame || p.iz == 0 || p.iz == P.nz - 1;
        if (!frame) return;
        // exact state in fp64 from the fp64 images of the tables is not available on the R path: evaluate in R
        R X[G::NX > 0 ? G::NX : 1], Y[G::NY > 0 ? G::NY : 1], Z[G::NZ > 0 ? G::NZ : 1], q[M], dQ[M];
        for (int e = 0; e < G::NX; ++e) X[e] = P.tabX[e * P.nx + p.ix];
        for (int e = 0; e < G::NY; ++e) Y[e] = P.tabY[e * P.ny + p.iy];
        for (int e = 0; e < G::NZ; ++e) Z[e] = P.tabZ[e * P.nz + p.iz];
        G::template exact<R>(P.mms, P.T, X, Y, Z, q);
        for (int k = 0; k < M; ++k) dQ[k] = q[k] - P.ref[k];
        typename Sys::Ctx ctx;
        load_aux<Sys, R>(ctx, P, node);
        Sys::setup(ctx, dQ, P);
        static_for<0, M>([&](auto K) {
            constexpr int k = decltype(K)::value;
            R F[D], S;
            Sys::template flux<k>(ctx, dQ, P, F, S);
            using L = Lattice<D>;
            f[tile_off(node, M * Q) + (k * Q) * TILE] = weight0<D, R>() * dQ[k];
            for (int a = 0; a < D; ++a) {
                const R h = R(0.5) * F[a];
                const long long op = gather == GATHER_PULL ? pull_offset(1 + 2 * a, p, P.nx, P.ny, P.nz) : 0LL;
                const long long om = gather == GATHER_PULL ? pull_offset(2 + 2 * a, p, P.nx, P.ny, P.nz) : 0LL;
                f[tile_off(node + op, M * Q) + (k * Q + 1 + 2 * a) * TILE] = R(L::w1) * dQ[k] + h;
                f[tile_off(node + om, M * Q) + (k * Q + 2 + 2 * a) * TILE] = R(L::w1) * dQ[k] - h;
            }
        });
    }
}

}  // namespace lbmk
