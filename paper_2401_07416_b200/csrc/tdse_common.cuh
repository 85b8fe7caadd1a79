// tdse_common.cuh -- shared device helpers for libtdse (sm_100a).
// Index convention: flat offset ((b*nz + k)*ny + j)*nx + i, x fastest (include/tdse.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tdse {

enum { BC_PERIODIC = 0, BC_DIRICHLET = 1 };

struct Grid {
    int nx, ny, nz, batch;
    int bcx, bcy, bcz;
    long long plane;   // nx*ny
    long long cells;   // nx*ny*nz
};

// 16-byte vector of `real`: float4-equivalent or double2-equivalent; copies compile to 128-bit ops.
template <typename real>
struct alignas(16) Pack {
    static constexpr int N = 16 / sizeof(real);
    real e[N];
};

__device__ __forceinline__ int wrap_index(int i, int n) {
    i %= n;
    return i < 0 ? i + n : i;
}

// Deterministic block-wide sum of doubles (warp shuffle tree, then warp 0 over per-warp sums).
// `scratch` must hold 32 doubles.  Result valid in thread 0.
__device__ __forceinline__ double block_sum(double v, double* scratch) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nwarps = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();   // scratch may be in use by a previous call
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < nwarps ? scratch[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

}  // namespace tdse
