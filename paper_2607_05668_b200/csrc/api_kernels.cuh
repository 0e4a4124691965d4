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

// plain streaming copy: the roofline denominator probe (cf. the paper's BabelStream peak)
__global__ void __launch_bounds__(256) copy_kernel(float4* __restrict__ dst, const float4* __restrict__ src, size_t n16) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

}  // namespace lbmk
