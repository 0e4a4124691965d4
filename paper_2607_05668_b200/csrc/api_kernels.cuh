// api_kernels.cuh -- system-independent kernels, compiled once (in lbmk_api.cu).
#pragma once
#include "common.cuh"

namespace lbmk {

// test hook: source node of direction `dir` for every node, through pull_offset
__global__ void stream_index_map_kernel(long long* __restrict__ out, int dir, int nx, int ny, int nz, long long n) {
    const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= n) return;
    const NodeIdx p = decompose(node, nx, ny);
    out[node] = node + pull_offset(dir, p, nx, ny, nz);
}

// Halo exchange of a slab: the slowest axis (z in 3D, y in 2D) carries one ghost plane at each
// end.  In the two-lattice pull storage (post-collision, stream pending) the next step of the first interior plane
// pulls slot(+s) from the lower ghost plane and the last interior plane pulls slot(-s) from the upper one; these
// are the ONLY ghost values the interior ever reads.  pack: buf[k][j] = slot `slot` of component k at node
// plane*plane_nodes + j; unpack: the inverse.  One thread per (k, j).
template <class R, bool PACK>
__global__ void halo_kernel(R* __restrict__ f, R* __restrict__ buf, int M, int Q, int slot, long long plane_first_node, long long plane_nodes) {
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (long long)M * plane_nodes) return;
    const int k = (int)(id / plane_nodes);
    const long long j = id - (long long)k * plane_nodes;
    const long long e = tile_off(plane_first_node + j, M * Q) + (long long)(k * Q + slot) * TILE;
    if (PACK) buf[id] = f[e]; else f[e] = buf[id];
}

// plain streaming copy: the roofline denominator probe (cf. the paper's BabelStream peak)
__global__ void __launch_bounds__(256) copy_kernel(float4* __restrict__ dst, const float4* __restrict__ src, size_t n16) {
    // one 16 KB chunk per block: 4 independent 128-bit loads per thread in flight, then 4 stores
    const size_t base = (size_t)blockIdx.x * 1024 + threadIdx.x;
    float4 v[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) if (base + 256 * j < n16) v[j] = src[base + 256 * j];
#pragma unroll
    for (int j = 0; j < 4; ++j) if (base + 256 * j < n16) dst[base + 256 * j] = v[j];
}

}  // namespace lbmk
