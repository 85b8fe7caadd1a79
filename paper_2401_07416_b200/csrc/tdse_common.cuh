// tdse_common.cuh -- shared device helpers for libtdse (sm_100a).
// Index convention of the C ABI (host buffers, include/tdse.h): flat offset ((b*nz + k)*ny + j)*nx + i, x fastest.
// Device storage of R, I, V adds a frame of PADX columns and PADY rows around every xy plane:
//   element (i, j, k) of entry b lives at  b*pcells + (k*py + j + PADY)*px + i + PADX,  px = nx + 2 PADX, py = ny + 2 PADY.
// On a periodic axis the frame holds the periodic images of the cells next to the opposite face (every kernel that
// writes a field writes the images too); on a Dirichlet axis it stays zero.  The fused kernel's TMA boxes (tile +
// halo) therefore never need index wrapping in x or y, and out-of-range z planes are zero-filled by the TMA unit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tdse {

enum { BC_PERIODIC = 0, BC_DIRICHLET = 1 };

constexpr int PADX = 4, PADY = 4;

struct Grid {
    int nx, ny, nz, batch;
    int bcx, bcy, bcz;
    int px, py;        // padded row length / rows per plane (elements)
    long long plane;   // nx*ny        (logical cells per plane)
    long long cells;   // nx*ny*nz     (logical cells per entry)
    long long pplane;  // px*py        (stored elements per plane)
    long long pcells;  // px*py*nz     (stored elements per entry)
};

// offset of logical cell (i, j, k) inside one entry's storage; i, j may reach into the frame
__host__ __device__ __forceinline__ long long cell_offset(const Grid& g, int i, int j, int k) {
    return ((long long)k * g.py + (j + PADY)) * g.px + (i + PADX);
}

// Store v at logical cell (i, j, k) and at its periodic images inside the frame.
template <typename real>
__device__ __forceinline__ void store_with_images(real* __restrict__ f, const Grid& g, int i, int j, int k, real v) {
    const long long o = cell_offset(g, i, j, k);
    f[o] = v;
    int ix = 0, jy = 0;                  // image shifts in cells (0: none)
    if (g.bcx == BC_PERIODIC) { if (i < PADX) ix = g.nx; else if (i >= g.nx - PADX) ix = -g.nx; }
    if (g.bcy == BC_PERIODIC) { if (j < PADY) jy = g.ny; else if (j >= g.ny - PADY) jy = -g.ny; }
    if (ix) f[o + ix] = v;
    if (jy) f[o + (long long)jy * g.px] = v;
    if (ix && jy) f[o + ix + (long long)jy * g.px] = v;
}

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
