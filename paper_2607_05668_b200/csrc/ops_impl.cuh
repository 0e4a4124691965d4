// ops_impl.cuh -- launches of the templated kernels for one system; included by each sys_*.cu.
#pragma once
#include <algorithm>
#include <climits>
#include <cstring>
#include <vector>

#include "kernels.cuh"
#include "ops.h"

namespace lbmk {

template <class R> __host__ inline KParams<R>& kp(GridCore& g);
template <> __host__ inline KParams<double>& kp<double>(GridCore& g) { return g.Pd; }
template <> __host__ inline KParams<float>& kp<float>(GridCore& g) { return g.Pf; }

// launch shape of the node kernel per system: threads per block, min blocks per SM (register cap)
template <template <class> class S, class R> struct Tune { static constexpr int BLOCK = 128, MINB = 1; };
#ifndef LBMK_NSF3D_BLOCK
#define LBMK_NSF3D_BLOCK 64
#endif
#ifndef LBMK_NSF3D_MINB
#define LBMK_NSF3D_MINB 6
#endif
template <class R> struct Tune<SysNsf3D, R> { static constexpr int BLOCK = LBMK_NSF3D_BLOCK, MINB = LBMK_NSF3D_MINB; };
template <> struct Tune<SysNsf3D, double> { static constexpr int BLOCK = 128, MINB = 1; };
template <class R> struct Tune<SysMhd3D, R> { static constexpr int BLOCK = 64, MINB = 4; };
template <class R> struct Tune<SysHcnsf3D, R> { static constexpr int BLOCK = 64, MINB = 6; };
template <> struct Tune<SysHcnsf3D, double> { static constexpr int BLOCK = 128, MINB = 1; };
template <class R> struct Tune<SysMhd2D, R> { static constexpr int BLOCK = 128, MINB = 3; };
template <> struct Tune<SysMhd2D, double> { static constexpr int BLOCK = 128, MINB = 1; };

// launch shape of the persistent kernel (L2-resident grids: latency-bound, so occupancy matters more than for the
// bandwidth-bound per-launch kernel)
#ifndef LBMK_P_BLOCK
#define LBMK_P_BLOCK 128
#endif
#ifndef LBMK_P_MINB
#define LBMK_P_MINB 1
#endif
template <template <class> class S, class R> struct TuneP { static constexpr int BLOCK = Tune<S, R>::BLOCK == 64 ? 64 : LBMK_P_BLOCK, MINB = Tune<S, R>::BLOCK == 64 ? Tune<S, R>::MINB : LBMK_P_MINB; };

// two-pass kernel: register cap via min blocks per SM
template <template <class> class S, class R> struct Tune2 { static constexpr int BLOCK = 256, MINB = 2; };
template <class R> struct Tune2<SysNsf3D, R> { static constexpr int BLOCK = 128, MINB = 4; };
template <class R> struct Tune2<SysMhd3D, R> { static constexpr int BLOCK = 128, MINB = 4; };
template <class R> struct Tune2<SysHcnsf3D, R> { static constexpr int BLOCK = 128, MINB = 4; };
template <class R> struct Tune2<SysMhd2D, R> { static constexpr int BLOCK = 128, MINB = 4; };

template <class Mm> struct MmsCounts { static constexpr int NT = Mm::NT, NX = Mm::NX, NY = Mm::NY, NZ = Mm::NZ, NC = Mm::NC; };
template <> struct MmsCounts<void> { static constexpr int NT = 0, NX = 0, NY = 0, NZ = 0, NC = 0; };

inline unsigned blocks_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

template <template <class> class S>
struct Ops {
    using Sd = S<double>;
    static constexpr int D = Sd::D, Q = 2 * D + 1, M = Sd::M;
    static constexpr bool HAS_MMS = has_mms<Sd>();
    static constexpr int NA = AuxCount<Sd>::value;

    using C = MmsCounts<typename Sd::Mms>;

    // ---- manufactured-solution tables and time scalars (host fp64)
    static void time_scalars(GridCore& g, double t) {
        if constexpr (HAS_MMS) {
            double T[8] = {0};
            Sd::Mms::time_scalars(t, g.mh, T);
            for (int i = 0; i < 8; ++i) { g.Pd.T[i] = T[i]; g.Pf.T[i] = (float)T[i]; }
        }
    }
    template <class R>
    static cudaError_t fill_tables_t(GridCore& g) {
        if constexpr (HAS_MMS) {
            const int cnt[3] = {C::NX, C::NY, C::NZ};
            const int len[3] = {g.nx, g.ny, g.nz};
            const int org[3] = {g.Pd.ox, g.Pd.oy, g.Pd.oz};
            for (int ax = 0; ax < 3; ++ax) {
                if (cnt[ax] == 0) continue;
                std::vector<R> h((size_t)cnt[ax] * len[ax]);
                double row[8];
                for (int j = 0; j < len[ax]; ++j) {
                    Sd::Mms::axis_row(ax, (j + org[ax]) * g.mh.dx, g.mh, row);   // x_j = j dx (reading A1), plus the sub-domain origin
                    for (int e = 0; e < cnt[ax]; ++e) h[(size_t)e * len[ax] + j] = (R)row[e];
                }
                cudaError_t e = cudaMemcpyAsync(g.tab[ax], h.data(), h.size() * sizeof(R), cudaMemcpyHostToDevice, g.stream);
                if (e != cudaSuccess) return e;
                e = cudaStreamSynchronize(g.stream);                         // h goes out of scope
                if (e != cudaSuccess) return e;
            }
            kp<R>(g).tabX = (const R*)g.tab[0]; kp<R>(g).tabY = (const R*)g.tab[1]; kp<R>(g).tabZ = (const R*)g.tab[2];
            kp<R>(g).coef = (const R*)g.coef;
        }
        kp<R>(g).aux = (const R*)g.aux_buf;
        kp<R>(g).aux_stride = g.aux_stride;
        kp<R>(g).node0 = 0;
        kp<R>(g).node1 = g.n;
        if (g.prec != PREC_F64) { g.Pd.node0 = 0; g.Pd.node1 = g.n; }
        return cudaSuccess;
    }
    static cudaError_t fill_tables(GridCore& g) { return g.prec == PREC_F64 ? fill_tables_t<double>(g) : fill_tables_t<float>(g); }

    static cudaError_t reference_equilibrium(GridCore& g) {
        KParams<double> P0 = g.Pd;
        for (int k = 0; k < MAXM; ++k) P0.ref[k] = 0.0;
        for (int k = 0; k < 8; ++k) P0.cst[k] = 0.0;
        reference_equilibrium_kernel<Sd><<<1, 1, 0, g.stream>>>(g.feq0, P0, g.Pd);
        g.launches++;
        return cudaGetLastError();
    }

    // nodes [node0, node1) from a buffer holding that range, component planes `ustride` apart; the last range ends the initialisation
    template <class R>
    static cudaError_t init_t(GridCore& g, const double* U, long long ustride, long long node0, long long node1) {
        init_from_U_kernel<S<R>, R><<<blocks_for(node1 - node0, 256), 256, 0, g.stream>>>(U, ustride, node0, node1, (R*)g.f[0], kp<R>(g), g.Pd);
        g.launches++;
        g.cur = 0;
        g.pending = 0;
        return cudaGetLastError();
    }
    static cudaError_t init_range(GridCore& g, const double* U, long long ustride, long long node0, long long node1) {
        return g.prec == PREC_F64 ? init_t<double>(g, U, ustride, node0, node1) : init_t<float>(g, U, ustride, node0, node1);
    }
    static cudaError_t init_from_U(GridCore& g, const double* U) { return init_range(g, U, g.n, 0, g.n); }

    template <class R>
    static cudaError_t set_f_t(GridCore& g, const double* f) {
        set_f_kernel<R><<<blocks_for(g.n, 256), 256, 0, g.stream>>>(f, (R*)g.f[0], g.feq0, M * Q, g.n);
        g.launches++;
        g.cur = 0;
        g.pending = 0;
        return cudaGetLastError();
    }
    static cudaError_t set_f(GridCore& g, const double* f) { return g.prec == PREC_F64 ? set_f_t<double>(g, f) : set_f_t<float>(g, f); }

    template <class R>
    static cudaError_t set_aux_t(GridCore& g, const double* A) {
        if constexpr (NA > 0) {
            set_aux_kernel<R><<<blocks_for(g.n, 256), 256, 0, g.stream>>>(A, (R*)g.aux_buf, NA, g.n, g.aux_stride);
            g.launches++;
            g.aux_set = true;
            return cudaGetLastError();
        }
        return cudaErrorNotSupported;
    }
    static cudaError_t set_aux(GridCore& g, const double* A) { return g.prec == PREC_F64 ? set_aux_t<double>(g, A) : set_aux_t<float>(g, A); }

    // where the canonical population sits in the current storage (kernels.cuh GATHER_*)
    static int aa_odd(const GridCore& g) {
        if (g.pattern == PATTERN_AA) return (g.step & 1) ? GATHER_AA_ODD : GATHER_CANON;
        return g.pending ? GATHER_PULL : GATHER_CANON;
    }

    template <class R>
    static cudaError_t read_U_t(GridCore& g, double* U, long long ustride, long long node0, long long node1) {
        read_U_kernel<Q, R><<<blocks_for(node1 - node0, 256), 256, 0, g.stream>>>((const R*)g.f[g.cur], U, ustride, node0, node1, M, g.nx, g.ny, g.nz,
                                                                                  aa_odd(g), g.Pd);
        g.launches++;
        return cudaGetLastError();
    }
    static cudaError_t read_range(GridCore& g, double* U, long long ustride, long long node0, long long node1) {
        return g.prec == PREC_F64 ? read_U_t<double>(g, U, ustride, node0, node1) : read_U_t<float>(g, U, ustride, node0, node1);
    }
    static cudaError_t read_U(GridCore& g, double* U) { return read_range(g, U, g.n, 0, g.n); }

    template <class R>
    static cudaError_t read_f_t(GridCore& g, double* f) {
        read_f_kernel<Q, R><<<blocks_for(g.n, 256), 256, 0, g.stream>>>((const R*)g.f[g.cur], f, g.feq0, M, g.nx, g.ny, g.nz, g.n, aa_odd(g));
        g.launches++;
        return cudaGetLastError();
    }
    static cudaError_t read_f(GridCore& g, double* f) { return g.prec == PREC_F64 ? read_f_t<double>(g, f) : read_f_t<float>(g, f); }

    template <class R>
    static cudaError_t wave_t(GridCore& g, double* out3) {
        cudaError_t e = cudaMemsetAsync(g.red, 0, 4 * sizeof(unsigned long long), g.stream);
        if (e != cudaSuccess) return e;
        const unsigned nb = (unsigned)std::min<long long>((g.n + 255) / 256, (long long)g.num_sms * 8);
        max_wave_speed_kernel<Sd, R><<<nb, 256, 0, g.stream>>>((const R*)g.f[g.cur], g.red, g.n, g.nx, g.ny, g.nz, aa_odd(g), g.Pd);
        g.launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        unsigned long long h[3];
        e = cudaMemcpyAsync(h, g.red, sizeof(h), cudaMemcpyDeviceToHost, g.stream);
        if (e != cudaSuccess) return e;
        e = cudaStreamSynchronize(g.stream);
        if (e != cudaSuccess) return e;
        for (int j = 0; j < 3; ++j) { double d; memcpy(&d, &h[j], 8); out3[j] = d; }
        return cudaSuccess;
    }
    static cudaError_t max_wave_speed(GridCore& g, double* out3) { return g.prec == PREC_F64 ? wave_t<double>(g, out3) : wave_t<float>(g, out3); }

    // ---- the step
    // launches over the node range [kp.node0, kp.node1) (whole grid unless step_ranges narrowed it)
    template <class R, int MODE, bool MMS>
    static void launch_node(GridCore& g, const R* src, R* dst, bool peer = false) {
        constexpr int BLOCK = Tune<S, R>::BLOCK, MINB = Tune<S, R>::MINB;
        const long long cnt = kp<R>(g).node1 - kp<R>(g).node0;
        if (cnt <= 0) return;
        if (peer) {                       // boundary planes of a slab with direct stores into the neighbours' ghost planes (BGK, node kernel)
            if constexpr (MODE == MODE_PULL2 || MODE == MODE_LOCAL)
                collide_stream_node<S<R>, R, MODE, MMS, BLOCK, MINB, false, true><<<blocks_for(cnt, BLOCK), BLOCK, 0, g.stream>>>(src, dst, kp<R>(g));
            g.launches++;
            return;
        }
        constexpr int NPT = 4;
        if constexpr (!MMS && M == 1 && NA == 0 && sizeof(R) == 4 && (MODE == MODE_PULL2 || MODE == MODE_LOCAL)) {
            // single-field fp32 systems: NPT nodes per thread for memory-level parallelism (kernels.cuh collide_stream_multi;
            // measured: Burgers 4096^2 fp32 154 -> 166 GLUPS = 94 % -> 101 % of the copy peak; fp64 already at 103 %: unchanged)
            if (g.collision == 0 && g.kernel == KERNEL_NODE && cnt >= (long long)BLOCK * NPT * g.num_sms) {
                collide_stream_multi<S<R>, R, MODE, BLOCK, NPT><<<blocks_for(cnt, BLOCK * NPT), BLOCK, 0, g.stream>>>(src, dst, kp<R>(g));
                g.launches++;
                return;
            }
        }
        if (g.collision == 1) {           // TRT: two-lattice modes of the node kernel only (checked at grid creation)
            if constexpr (MODE == MODE_PULL2 || MODE == MODE_LOCAL)
                collide_stream_node<S<R>, R, MODE, MMS, BLOCK, MINB, true><<<blocks_for(cnt, BLOCK), BLOCK, 0, g.stream>>>(src, dst, kp<R>(g));
        } else if (g.kernel == KERNEL_TWOPASS) {
            constexpr int B2 = Tune2<S, R>::BLOCK, M2 = Tune2<S, R>::MINB;
            collide_stream_twopass<S<R>, R, MODE, MMS, B2, M2><<<blocks_for(cnt, B2), B2, 0, g.stream>>>(src, dst, kp<R>(g));
        } else {
            collide_stream_node<S<R>, R, MODE, MMS, BLOCK, MINB><<<blocks_for(cnt, BLOCK), BLOCK, 0, g.stream>>>(src, dst, kp<R>(g));
        }
        g.launches++;
    }
    // ---- persistent stepping: `cnt` steps of the two-lattice pull pattern in ONE cooperative launch (kernels.cuh)
    template <class R, bool MMS>
    static int persistent_grid(GridCore& g, int* rounds_out = nullptr) {
        constexpr int BLOCK = TuneP<S, R>::BLOCK, MINB = TuneP<S, R>::MINB;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, collide_stream_persistent<S<R>, R, MMS, BLOCK, MINB>, BLOCK, 0) != cudaSuccess) return 0;
        const long long cap = std::min<long long>((long long)per_sm * g.num_sms, PERSISTENT_MAX_BLOCKS), nseg = (g.n + BLOCK - 1) / BLOCK;
        if (cap <= 0) return 0;
        const long long rounds = (nseg + cap - 1) / cap;          // segments per block and step
        if (rounds > INT_MAX) return 0;
        if (rounds_out) *rounds_out = (int)rounds;
        return (int)((nseg + rounds - 1) / rounds);               // balanced: every block owns `rounds` consecutive segments (the last one fewer)
    }
    // fat blocks (kernels.cuh collide_stream_persistent_fat): 4 x 128 threads, one block per SM, when every block then owns at least
    // FAT_MIN_ROUNDS segments (so that it has an interior to hide the flag round trip behind) and the coefficients are unstaged
#ifndef LBMK_FAT_GROUPS
#define LBMK_FAT_GROUPS 4
#endif
    static constexpr int FAT_GROUPS = LBMK_FAT_GROUPS, FAT_MIN_ROUNDS = 8;
    template <class R, bool MMS>
    static constexpr bool fat_capable() {      // <= 160 B of populations per node: fits the 128 registers of a 512-thread block without spilling
        return TuneP<S, R>::BLOCK == 128 && !(MMS && C::NC >= STAGE_MIN_NC) && (size_t)M * Q * sizeof(R) <= 160;
    }
    template <class R, bool MMS>
    static int persistent_fat_grid(GridCore& g, int* rounds_out) {
        if constexpr (fat_capable<R, MMS>()) {
            constexpr int BLOCK = 128;
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, collide_stream_persistent_fat<S<R>, R, MMS, BLOCK, FAT_GROUPS>, BLOCK * FAT_GROUPS, 0) != cudaSuccess) return 0;
            const long long cap = std::min<long long>((long long)(per_sm > 0 ? 1 : 0) * g.num_sms, PERSISTENT_MAX_BLOCKS), nseg = (g.n + BLOCK - 1) / BLOCK;
            if (cap <= 0) return 0;
            const long long rounds = (nseg + cap - 1) / cap;
            if (rounds < FAT_MIN_ROUNDS || rounds > INT_MAX) return 0;
            *rounds_out = (int)rounds;
            return (int)((nseg + rounds - 1) / rounds);
        }
        return 0;
    }
    template <class R, bool MMS>
    static cudaError_t launch_persistent(GridCore& g, int cnt, long long coef_stride) {
        constexpr int BLOCK = TuneP<S, R>::BLOCK, MINB = TuneP<S, R>::MINB;
        int rounds = 0;
        bool fat = true;
        int grid = persistent_fat_grid<R, MMS>(g, &rounds);
        if (grid <= 0) { fat = false; grid = persistent_grid<R, MMS>(g, &rounds); }
        if (grid <= 0) return cudaErrorLaunchOutOfResources;
        cudaError_t e = cudaMemsetAsync(g.bar, 0, (size_t)grid * FLAG_STRIDE * sizeof(unsigned int), g.stream);     // one "steps done" flag per block
        if (e != cudaSuccess) return e;
        R* fa = (R*)g.f[g.cur];
        R* fb = (R*)g.f[g.cur ^ 1];
        KParams<R> P = kp<R>(g);
        int first_local = g.pending ? 0 : 1;
        unsigned int* bar = g.bar;
        void* args[] = {&fa, &fb, &P, &cnt, &first_local, &coef_stride, &bar, &rounds};
        if constexpr (fat_capable<R, MMS>()) {
            if (fat) e = cudaLaunchCooperativeKernel((const void*)collide_stream_persistent_fat<S<R>, R, MMS, 128, FAT_GROUPS>, dim3(grid), dim3(128 * FAT_GROUPS), args, 0, g.stream);
        }
        if (!fat) e = cudaLaunchCooperativeKernel((const void*)collide_stream_persistent<S<R>, R, MMS, BLOCK, MINB>, dim3(grid), dim3(BLOCK), args, 0, g.stream);
        if (e != cudaSuccess) return e;
        g.launches++;
        g.persistent_launches++;
        g.cur ^= (cnt & 1);
        g.pending = 1;
        g.step += cnt;
        return cudaSuccess;
    }
    // ---- SM-resident stepping: ONE population copy in the shared memory of all SMs, AA pattern in place (kernels.cuh)
    static constexpr size_t RESIDENT_SMEM_MAX = 227 * 1024;
    template <class R> struct TuneR { static constexpr int BLOCK = (size_t)M * Q * sizeof(R) <= 160 ? 512 : 256; };
    template <class R>
    static int resident_rounds(const GridCore& g) {         // tiles per block, or 0 if the grid does not fit
        if (g.num_sms <= 0) return 0;
        const long long ntile = (g.n + TILE - 1) / TILE;
        const long long rounds = (ntile + g.num_sms - 1) / g.num_sms;
        const size_t smem = (size_t)rounds * M * Q * TILE * sizeof(R);
        return (smem <= RESIDENT_SMEM_MAX && rounds <= INT_MAX) ? (int)rounds : 0;
    }
    static bool resident_supported(const GridCore& g) { return (g.prec == PREC_F64 ? resident_rounds<double>(g) : resident_rounds<float>(g)) > 0; }
    template <class R, bool MMS>
    static cudaError_t launch_resident(GridCore& g, int cnt, long long coef_stride) {
        constexpr int BLOCK = TuneR<R>::BLOCK;
        int rounds = resident_rounds<R>(g);
        if (rounds <= 0) return cudaErrorLaunchOutOfResources;
        const long long ntile = (g.n + TILE - 1) / TILE;
        const int grid = (int)((ntile + rounds - 1) / rounds);
        const size_t smem = (size_t)rounds * M * Q * TILE * sizeof(R);
        auto kern = collide_stream_resident<S<R>, R, MMS, BLOCK>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(g.bar, 0, (size_t)grid * FLAG_STRIDE * sizeof(unsigned int), g.stream);
        if (e != cudaSuccess) return e;
        R* f = (R*)g.f[0];
        KParams<R> P = kp<R>(g);
        int parity0 = (int)(g.step & 1);
        unsigned int* bar = g.bar;
        void* args[] = {&f, &P, &cnt, &parity0, &coef_stride, &bar, &rounds};
        e = cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(BLOCK), args, smem, g.stream);
        if (e != cudaSuccess) return e;
        g.launches++;
        g.persistent_launches++;
        g.step += cnt;
        return cudaSuccess;
    }
    static bool use_resident(const GridCore& g, int n_steps) {
        return g.stepping == STEPPING_RESIDENT && g.pattern == PATTERN_AA && g.kernel == KERNEL_NODE && g.bc == 0 && g.collision == 0 && n_steps >= 2;
    }
    // ---- cluster-resident stepping for tiny grids: state in distributed shared memory of one cluster (kernels.cuh)
    static constexpr int CLUSTER = 8;
    template <class R>
    static int cluster_npc(const GridCore& g) {        // threads (= nodes) per CTA, or 0 if the grid does not qualify
        if (HAS_MMS && g.mms_id != 0) return 0;
        if (NA > 0 || M * Q > 40 || g.n > (long long)CLUSTER * 1024 || g.n < 64) return 0;   // small tracker-free systems (<= 64 registers at 1024 threads)
        const int npc = (int)(((g.n + CLUSTER - 1) / CLUSTER + 31) / 32 * 32);
        const size_t smem = 2 * (size_t)M * Q * npc * sizeof(R);
        return smem <= (size_t)200 * 1024 ? npc : 0;
    }
    template <class R>
    static cudaError_t launch_cluster(GridCore& g, int cnt, int npc) {
        const size_t smem = 2 * (size_t)M * Q * npc * sizeof(R);
        auto kern = collide_stream_cluster<S<R>, R>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(CLUSTER); cfg.blockDim = dim3(npc); cfg.dynamicSmemBytes = smem; cfg.stream = g.stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = CLUSTER; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        const R* src = (const R*)g.f[g.cur];
        R* dst = (R*)g.f[g.cur ^ 1];
        e = cudaLaunchKernelEx(&cfg, kern, src, dst, kp<R>(g), cnt, g.pending ? 0 : 1);
        if (e != cudaSuccess) return e;
        g.launches++;
        g.persistent_launches++;
        g.cur ^= 1;                       // whatever cnt: the result is in the other buffer
        g.pending = 1;
        g.step += cnt;
        return cudaSuccess;
    }
    static bool cluster_supported(const GridCore& g) { return (g.prec == PREC_F64 ? cluster_npc<double>(g) : cluster_npc<float>(g)) > 0; }
    static bool use_persistent(const GridCore& g, int n_steps) {
        return (g.stepping == STEPPING_PERSISTENT || g.stepping == STEPPING_CLUSTER) && g.pattern == PATTERN_PULL2 && g.kernel == KERNEL_NODE && g.bc == 0 && n_steps >= 2;
    }
    // one collide-and-stream launch (plus the Dirichlet frame refill before it on bounded grids)
    template <class R, bool MMS>
    static void one_step(GridCore& g) {
        if (g.bc == 1) {
            if constexpr (HAS_MMS) {
                time_scalars(g, g.t0 + (double)g.step * g.dt);
                dirichlet_frame_kernel<S<R>, R><<<blocks_for(g.n, 256), 256, 0, g.stream>>>((R*)g.f[g.cur], aa_odd(g), kp<R>(g), g.Pd);
                g.launches++;
            }
        }
        if (g.pattern == PATTERN_PULL2) {
            if (g.pending) launch_node<R, MODE_PULL2, MMS>(g, (const R*)g.f[g.cur], (R*)g.f[g.cur ^ 1]);
            else launch_node<R, MODE_LOCAL, MMS>(g, (const R*)g.f[g.cur], (R*)g.f[g.cur ^ 1]);
            g.cur ^= 1;
            g.pending = 1;
        } else if ((g.step & 1) == 0) {
            launch_node<R, MODE_AA_EVEN, MMS>(g, (const R*)g.f[0], (R*)g.f[0]);
        } else {
            launch_node<R, MODE_AA_ODD, MMS>(g, (const R*)g.f[0], (R*)g.f[0]);
        }
        g.step++;
    }
    // row coefficients of steps [first, first + nb) into coefficient buffer `buf`, on the auxiliary stream
    template <class R>
    static void launch_coeffs(GridCore& g, int buf, long long first, int nb) {
        const long long rows = (long long)g.ny * g.nz;
        R* dst = (R*)g.coef + (size_t)buf * g.coef_B * rows * C::NC;
        const long long threads = rows * nb;
        mms_row_coeffs_kernel<S<R>, R><<<(unsigned)((threads + 127) / 128), 128, 0, g.aux>>>(
            dst, g.ny, g.nz, g.Pd.oy, g.Pd.oz, nb, g.t0 + (double)first * g.dt, g.dt, g.mh, g.Pd.mms);
        g.launches++;
    }
    template <class R, bool MMS>
    static cudaError_t step_t(GridCore& g, int n_steps) {
        if constexpr (!MMS) {
            if (use_resident(g, n_steps)) {
                for (int done = 0; done < n_steps;) {
                    const int cnt = std::min(n_steps - done, 1 << 16);
                    cudaError_t e = launch_resident<R, false>(g, cnt, 0);
                    if (e != cudaSuccess) return e;
                    done += cnt;
                }
                return cudaGetLastError();
            }
            if (use_persistent(g, n_steps)) {
                if (g.stepping == STEPPING_CLUSTER) return launch_cluster<R>(g, n_steps, cluster_npc<R>(g));
                for (int done = 0; done < n_steps;) {
                    const int cnt = std::min(n_steps - done, 1 << 16);      // bounds the 32-bit barrier count
                    cudaError_t e = launch_persistent<R, false>(g, cnt, 0);
                    if (e != cudaSuccess) return e;
                    done += cnt;
                }
                return cudaGetLastError();
            }
            for (int s = 0; s < n_steps; ++s) one_step<R, false>(g);
            return cudaGetLastError();
        } else {
            // Explicit forcing at the temporal midpoint (L154).  Its per-row coefficients are produced in batches of
            // coef_B steps on the auxiliary stream, double-buffered: batch j+1 is computed while batch j is consumed.
            const long long rows = (long long)g.ny * g.nz;
            const int B = g.coef_B;
            cudaError_t e = cudaEventRecord(g.ev_entry, g.stream);       // earlier calls may still read the buffers
            if (e != cudaSuccess) return e;
            e = cudaStreamWaitEvent(g.aux, g.ev_entry, 0);
            if (e != cudaSuccess) return e;
            int done = 0, buf = 0;
            launch_coeffs<R>(g, 0, g.step, std::min(B, n_steps));
            cudaEventRecord(g.ev_coef[0], g.aux);
            g.coef_used[0] = g.coef_used[1] = false;
            while (done < n_steps) {
                const int cnt = std::min(B, n_steps - done);
                if (done + cnt < n_steps) {
                    if (g.coef_used[buf ^ 1]) cudaStreamWaitEvent(g.aux, g.ev_free[buf ^ 1], 0);
                    launch_coeffs<R>(g, buf ^ 1, g.step + cnt, std::min(B, n_steps - done - cnt));
                    cudaEventRecord(g.ev_coef[buf ^ 1], g.aux);
                }
                e = cudaStreamWaitEvent(g.stream, g.ev_coef[buf], 0);
                if (e != cudaSuccess) return e;
                if (use_resident(g, cnt)) {
                    kp<R>(g).coef = (const R*)g.coef + (size_t)buf * B * rows * C::NC;
                    e = launch_resident<R, true>(g, cnt, rows * C::NC);
                    if (e != cudaSuccess) return e;
                } else if (use_persistent(g, cnt)) {          // the whole batch of steps in one cooperative launch
                    kp<R>(g).coef = (const R*)g.coef + (size_t)buf * B * rows * C::NC;
                    e = launch_persistent<R, true>(g, cnt, rows * C::NC);
                    if (e != cudaSuccess) return e;
                } else {
                    for (int j = 0; j < cnt; ++j) {
                        kp<R>(g).coef = (const R*)g.coef + ((size_t)buf * B + j) * rows * C::NC;
                        one_step<R, true>(g);
                    }
                }
                cudaEventRecord(g.ev_free[buf], g.stream);
                g.coef_used[buf] = true;
                done += cnt;
                buf ^= 1;
            }
            return cudaGetLastError();
        }
    }
    static cudaError_t step(GridCore& g, int n_steps) {
        const bool mms = HAS_MMS && g.mms_id != 0;
        if constexpr (HAS_MMS) {
            if (mms) return g.prec == PREC_F64 ? step_t<double, true>(g, n_steps) : step_t<float, true>(g, n_steps);
        }
        return g.prec == PREC_F64 ? step_t<double, false>(g, n_steps) : step_t<float, false>(g, n_steps);
    }
    // One step of a slab split into its boundary planes (two ranges) and its interior (third range): the boundary ranges
    // go first and `ev` marks their completion, so that the halo exchange can run while the interior is updated.
    template <class R, bool MMS>
    static cudaError_t step_ranges_t(GridCore& g, const long long* r, cudaEvent_t ev, int peer) {
        if (g.pattern != PATTERN_PULL2 || g.bc != 0) return cudaErrorNotSupported;
        if (peer) {
            if (!g.peers_set || g.collision != 0 || g.kernel != KERNEL_NODE) return cudaErrorNotSupported;
            const long long pn = D == 3 ? (long long)g.nx * g.ny : (long long)g.nx;
            const int np = D == 3 ? g.nz : g.ny;
            KParams<R>& P = kp<R>(g);
            P.peer_lo = (R*)g.peer_f[0][g.cur ^ 1]; P.peer_hi = (R*)g.peer_f[1][g.cur ^ 1];     // the neighbours' destination buffers of this step
            P.peer_lo_node0 = g.peer_node0[0]; P.peer_hi_node0 = g.peer_node0[1];
            P.plane_nodes = pn; P.last_own0 = (long long)(np - 2) * pn;
        }
        const int buf = (int)(g.step & 1);
        if constexpr (MMS) {
            // this step's row coefficients on the auxiliary stream, double-buffered by step parity: the pre-kernel of
            // step s runs under the kernels of step s-1
            const long long rows = (long long)g.ny * g.nz;
            cudaError_t e = cudaSuccess;
            if (g.coef_used[buf]) e = cudaStreamWaitEvent(g.aux, g.ev_free[buf], 0);
            else { e = cudaEventRecord(g.ev_entry, g.stream); if (e == cudaSuccess) e = cudaStreamWaitEvent(g.aux, g.ev_entry, 0); }
            if (e != cudaSuccess) return e;
            launch_coeffs<R>(g, buf, g.step, 1);
            cudaEventRecord(g.ev_coef[buf], g.aux);
            e = cudaStreamWaitEvent(g.stream, g.ev_coef[buf], 0);
            if (e != cudaSuccess) return e;
            kp<R>(g).coef = (const R*)g.coef + (size_t)buf * g.coef_B * rows * C::NC;
        }
        const R* src = (const R*)g.f[g.cur];
        R* dst = (R*)g.f[g.cur ^ 1];
        for (int q = 0; q < 3; ++q) {
            kp<R>(g).node0 = r[2 * q]; kp<R>(g).node1 = r[2 * q + 1];
            if (g.pending) launch_node<R, MODE_PULL2, MMS>(g, src, dst, peer && q < 2);
            else launch_node<R, MODE_LOCAL, MMS>(g, src, dst, peer && q < 2);
            if (q == 1 && ev) cudaEventRecord(ev, g.stream);
        }
        kp<R>(g).node0 = 0; kp<R>(g).node1 = g.n;
        if constexpr (MMS) { cudaEventRecord(g.ev_free[buf], g.stream); g.coef_used[buf] = true; }
        g.cur ^= 1;
        g.pending = 1;
        g.step++;
        return cudaGetLastError();
    }
    static cudaError_t step_ranges(GridCore& g, const long long* r, cudaEvent_t ev, int peer) {
        const bool mms = HAS_MMS && g.mms_id != 0;
        if constexpr (HAS_MMS) {
            if (mms) return g.prec == PREC_F64 ? step_ranges_t<double, true>(g, r, ev, peer) : step_ranges_t<float, true>(g, r, ev, peer);
        }
        return g.prec == PREC_F64 ? step_ranges_t<double, false>(g, r, ev, peer) : step_ranges_t<float, false>(g, r, ev, peer);
    }
    // Dirichlet frame refresh before readback (the oracle does the same in orc_read_U)
    static cudaError_t frame_now(GridCore& g) {
        if constexpr (HAS_MMS) {
            if (g.bc == 1) {
                time_scalars(g, g.t0 + (double)g.step * g.dt);
                if (g.prec == PREC_F64) dirichlet_frame_kernel<S<double>, double><<<blocks_for(g.n, 256), 256, 0, g.stream>>>((double*)g.f[g.cur], aa_odd(g), g.Pd, g.Pd);
                else dirichlet_frame_kernel<S<float>, float><<<blocks_for(g.n, 256), 256, 0, g.stream>>>((float*)g.f[g.cur], aa_odd(g), g.Pf, g.Pd);
                g.launches++;
            }
        }
        return cudaGetLastError();
    }
    static cudaError_t read_U_with_frame(GridCore& g, double* U) {
        cudaError_t e = frame_now(g);
        if (e != cudaSuccess) return e;
        return read_U(g, U);
    }
    template <class R>
    static cudaError_t norms_t(GridCore& g, double* out) {
        cudaError_t e = cudaMemsetAsync(out, 0, (size_t)M * 6 * sizeof(double), g.stream);
        if (e != cudaSuccess) return e;
        const unsigned nb = (unsigned)std::min<long long>((g.n + 255) / 256, (long long)g.num_sms * 4);
        error_norms_kernel<Sd, R><<<nb, 256, 0, g.stream>>>((const R*)g.f[g.cur], out, g.n, g.nx, g.ny, g.nz, aa_odd(g),
                                                            g.t0 + (double)g.step * g.dt, g.mh, g.Pd);
        g.launches++;
        return cudaGetLastError();
    }
    static cudaError_t error_norms(GridCore& g, double* out) {
        if constexpr (!HAS_MMS) return cudaErrorNotSupported;
        cudaError_t e = frame_now(g);
        if (e != cudaSuccess) return e;
        return g.prec == PREC_F64 ? norms_t<double>(g, out) : norms_t<float>(g, out);
    }
    // the same norms through `scratch` ([nrec][M][6] doubles, nrec = ceil(n / NORM_RECORD_NODES)) into out_dev [M][6]; no atomics
    template <class R>
    static cudaError_t norm_records_t(GridCore& g, double* scratch, double* out_dev) {
        const long long nrec = (g.n + NORM_RECORD_NODES - 1) / NORM_RECORD_NODES;
        error_norm_records_kernel<Sd, R><<<(unsigned)nrec, 256, 0, g.stream>>>((const R*)g.f[g.cur], scratch, g.n, g.nx, g.ny, g.nz, aa_odd(g),
                                                                              g.t0 + (double)g.step * g.dt, g.mh, g.Pd);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        combine_norm_records_kernel<<<1, 128, 0, g.stream>>>(scratch, nrec, M * 6, out_dev);
        g.launches += 2;
        return cudaGetLastError();
    }
    static cudaError_t error_norm_records(GridCore& g, double* scratch, double* out_dev) {
        if constexpr (!HAS_MMS) return cudaErrorNotSupported;
        cudaError_t e = frame_now(g);
        if (e != cudaSuccess) return e;
        return g.prec == PREC_F64 ? norm_records_t<double>(g, scratch, out_dev) : norm_records_t<float>(g, scratch, out_dev);
    }
    using Gen = typename GenOf<S>::type;
    static constexpr bool HAS_GEN = !std::is_void<Gen>::value;
    template <class R>
    static cudaError_t selfcheck_t(GridCore& g, double g_tau, double* out_host) {
        if constexpr (HAS_GEN) {
            cudaError_t e = cudaMemsetAsync(g.red, 0, sizeof(unsigned long long), g.stream);
            if (e != cudaSuccess) return e;
            GenArgs<double> ga;
            for (int i = 0; i < 8; ++i) ga.par[i] = g.Pd.par[i];
            ga.dx = g.mh.dx; ga.dt = g.dt; ga.gtau = g_tau;
            const unsigned nb = (unsigned)std::min<long long>((g.n + 127) / 128, (long long)g.num_sms * 8);
            flux_selfcheck_kernel<Sd, Gen, R><<<nb, 128, 0, g.stream>>>((const R*)g.f[g.cur], (const R*)g.aux_buf, g.aux_stride, g.red, g.n,
                                                                        g.nx, g.ny, g.nz, aa_odd(g), g.Pd, ga);
            g.launches++;
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            unsigned long long h = 0;
            e = cudaMemcpyAsync(&h, g.red, sizeof(h), cudaMemcpyDeviceToHost, g.stream);
            if (e != cudaSuccess) return e;
            e = cudaStreamSynchronize(g.stream);
            if (e != cudaSuccess) return e;
            memcpy(out_host, &h, 8);
            return cudaSuccess;
        }
        return cudaErrorNotSupported;
    }
    static cudaError_t flux_selfcheck(GridCore& g, double g_tau, double* out_host) {
        return g.prec == PREC_F64 ? selfcheck_t<double>(g, g_tau, out_host) : selfcheck_t<float>(g, g_tau, out_host);
    }
    static bool row_supported(const GridCore&) { return false; }

    static const SysOps* get() {
        static const SysOps ops = {Sd::ID, D, M, Sd::MC, HAS_MMS, C::NT, {C::NX, C::NY, C::NZ}, C::NC, NA, IsLinear<Sd>::value,
                                   &fill_tables, &reference_equilibrium, &init_from_U, &set_f, &step, &step_ranges, &set_aux,
                                   &read_U_with_frame, &read_f, &max_wave_speed, &error_norms, &row_supported, &cluster_supported, HAS_GEN, &flux_selfcheck, &resident_supported, &init_range, &read_range, &frame_now, &error_norm_records};
        return &ops;
    }
};

}  // namespace lbmk
