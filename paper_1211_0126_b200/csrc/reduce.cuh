// reduce.cuh -- deterministic two-stage reductions (reading A19): every block writes one
// partial per source, the last block to arrive (atomic ticket) sums them in a fixed order.
#pragma once
#include "tsm_internal.cuh"

// Sum over ALL threads of the block (any blockDim.x * blockDim.y multiple of 32, <= 1024).
// Result valid in flat thread 0.  smem: >= 32 doubles.
__device__ __forceinline__ double block_sum_all(double v, double* smem)
{
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int nw = (blockDim.x * blockDim.y) >> 5;
    v = warp_sum(v);
    if ((tid & 31) == 0) smem[tid >> 5] = v;
    __syncthreads();
    double t = 0;
    if (tid == 0)
        for (int k = 0; k < nw; k++) t += smem[k];
    __syncthreads();
    return t;
}

// Call after the block's partials are written (by any of its threads).  Returns true, in every
// thread, for exactly one block of the grid: the last one to get here.  That block may then
// read all partials with __ldcg.  The ticket is reset for the next launch.
__device__ __forceinline__ bool last_block_arrive(unsigned* ticket)
{
    __shared__ int is_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0) {
        const unsigned total = gridDim.x * gridDim.y * gridDim.z;
        const unsigned t = atomicAdd(ticket, 1u);
        is_last = (t == total - 1);
        if (is_last) *ticket = 0;
    }
    __syncthreads();
    if (is_last) __threadfence();
    return is_last != 0;
}

// In the last block: total of partials[rhs * nblk + 0 .. nblk), summed by ONE warp (lane-strided,
// then the fixed shuffle tree), so the order depends on nblk only -- not on the block shape or on
// how many sources are in the batch (A14: a source's iterate is bit-identical in any batch).
// Call with all 32 lanes of the warp; result valid in lane 0.
__device__ __forceinline__ double sum_partials_warp(const double* partials, int rhs, int nblk)
{
    const int lane = (threadIdx.y * blockDim.x + threadIdx.x) & 31;
    double v = 0;
    for (int k = lane; k < nblk; k += 32) v += __ldcg(partials + (size_t)rhs * nblk + k);
    return warp_sum(v);
}
