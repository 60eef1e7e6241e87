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

// What follows the sum v of a stencil epilogue's partials for source rhs (O5; one thread):
//   which == 0 (after w = Mhat p, EPI_NORM):  pq = |w|^2 = Re<p,q>;  alpha = rr / pq, or 0 for a frozen
//              source; 0 / non-finite pq or rr freezes the source and flags TSM_EBREAKDOWN (A13)
//   which == 1 (after r -= alpha q, EPI_RESID): rr_new = |r|^2
__device__ __forceinline__ void cg_after_reduction(int which, int rhs, double v, CgScalars* cg)
{
    if (which == 1) { cg->rr_new[rhs] = v; return; }
    cg->pq[rhs] = v;
    double alpha = 0.0;
    if (!cg->done[rhs]) {
        const double rr = cg->rr[rhs];
        if (!(v > 0) || !isfinite(v) || !(rr > 0) || !isfinite(rr)) {
            cg->done[rhs] = 1;
            cg->status[rhs] = TSM_EBREAKDOWN;
            cg->sticky_breakdown = 1;
        } else {
            alpha = rr / v;
        }
    }
    cg->alpha[rhs] = alpha;
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
