// block_ops.cuh -- CTA-wide scan / reduction helpers shared by update.cu and chain_step.cu.
#pragma once
#include "bd_internal.cuh"

// Block-wide inclusive scan of three running sums over a chunk of blockDim.x items, plus carry-in.
// s_warp: [3][32] scratch.  Returns the inclusive prefix for this thread; `carry` (per-thread copy of the
// block-uniform running total) is advanced by the chunk total.
__device__ __forceinline__ void block_scan3(double& x, double& y, double& z, double* s_warp, double carry[3])
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        double tx = __shfl_up_sync(0xffffffffu, x, o);
        double ty = __shfl_up_sync(0xffffffffu, y, o);
        double tz = __shfl_up_sync(0xffffffffu, z, o);
        if (lane >= o) { x += tx; y += ty; z += tz; }
    }
    __syncthreads();                       // protect s_warp from the previous chunk's readers
    if (lane == 31) { s_warp[warp] = x; s_warp[32 + warp] = y; s_warp[64 + warp] = z; }
    __syncthreads();
    double ox = carry[0], oy = carry[1], oz = carry[2];
    for (int w = 0; w < warp; ++w) { ox += s_warp[w]; oy += s_warp[32 + w]; oz += s_warp[64 + w]; }
    x += ox; y += oy; z += oz;
    double tx = 0, ty = 0, tz = 0;
    for (int w = 0; w < nwarp; ++w) { tx += s_warp[w]; ty += s_warp[32 + w]; tz += s_warp[64 + w]; }
    carry[0] += tx; carry[1] += ty; carry[2] += tz;
}

__device__ __forceinline__ double block_sum(double x, double* s_red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    x = warp_sum(x);
    __syncthreads();
    if (lane == 0) s_red[warp] = x;
    __syncthreads();
    double t = 0;
    for (int w = 0; w < nwarp; ++w) t += s_red[w];
    return t;
}

