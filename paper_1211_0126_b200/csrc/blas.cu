// blas.cu -- H6: the fused BLAS-1 / reduction kernels of CG on Mhat^dag Mhat (O5).
//
// Per iteration (api_solve.cu: cg_iteration):
//   stencil 2 leaves |w|^2 = Re<p,q> per tile   -> k_cg_reduce(0): alpha = rr / Re<p,q>
//   stencil 4 does r -= alpha q, |r|^2 per tile  -> k_cg_reduce(1): rr' = |r|^2
//   k_cg_update_xp : x += alpha p; p = r + (rr'/rr) p   (one pass over x, p, r)
//                    last block: iteration count, stopping test |r|/|b'| <= tol (A8), freeze flags
// All scalars stay on the device (CgScalars); every source has its own (A14) and a finished
// source is frozen: its x, r, p are no longer touched.  Sums are deterministic (A19).
//
// PV is the storage precision of x, r, q; PP that of p (bf16 mode keeps x, r, q in fp32).
#include "reduce.cuh"

namespace {

constexpr int BLAS_BS = 256;

template <int PV, int PP>
__global__ void __launch_bounds__(BLAS_BS) k_cg_init(const int Vh, const int nrhs, const void* __restrict__ r_, void* __restrict__ p_,
                                                     void* __restrict__ x_, double* __restrict__ partials, CgScalars* cg)
{
    using TV = typename PT<PV>::real;
    using TP = typename PT<PP>::real;
    const int rhs = blockIdx.y;
    const char* r = (const char*)r_ + field_bytes(PV, Vh, 1) * rhs;
    char* x = (char*)x_ + field_bytes(PV, Vh, 1) * rhs;
    char* p = (char*)p_ + field_bytes(PP, Vh, 1) * rhs;
    double sum = 0;
    const int n = 3 * (int)padded_sites(Vh);
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += gridDim.x * blockDim.x) {
        const int k8 = (idx >> 5) % 3, i = (idx >> 5) / 3 * LB + (idx & 31);   // (layout block, k8, site in block)
        if (i >= Vh) continue;
        TV rv[8], z[8];
        TP pv[8];
        load8<PV>(r, i, k8, rv);
#pragma unroll
        for (int k = 0; k < 8; k++) { sum = fma((double)rv[k], (double)rv[k], sum); pv[k] = (TP)rv[k]; z[k] = 0; }   // explicit: k_cg_persistent_small repeats this chain
        store8<PP>(p, i, k8, pv);
        store8<PV>(x, i, k8, z);
    }
    __shared__ double smem[32];
    const double tot = block_sum_all(sum, smem);
    if (threadIdx.x == 0) partials[(size_t)rhs * gridDim.x + blockIdx.x] = tot;
    if (last_block_arrive(&cg->ticket)) {
        for (int j = threadIdx.x >> 5; j < nrhs; j += BLAS_BS / 32) {
            const double v = sum_partials_warp(partials, j, gridDim.x);
            if ((threadIdx.x & 31) == 0) {
                cg->rr[j] = v;
                cg->bb[j] = v;
                cg->pq[j] = 0;
                cg->beta[j] = 0;
                cg->iters[j] = 0;
                cg->status[j] = TSM_OK;
                cg->done[j] = !(v > 0);
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int all = 1;
            for (int j = 0; j < nrhs; j++) all &= cg->done[j];
            cg->all_done = all;
        }
    }
}

// Sum of the per-tile partials a stencil epilogue left for every source (one block per source; the order
// depends on ntiles only, so a source gets the same sum in any batch, A14/A19), then:
//   which == 0 (after w = Mhat p, EPI_NORM):  pq = |w|^2 = Re<p,q>;  alpha = rr / pq, or 0 for a frozen
//              source; 0 / non-finite pq or rr freezes the source and flags TSM_EBREAKDOWN (A13)
//   which == 1 (after r -= alpha q, EPI_RESID): rr_new = |r|^2
__global__ void __launch_bounds__(BLAS_BS) k_cg_reduce(const int which, const int force, const double* __restrict__ norm_partials,
                                                       const int ntiles, CgScalars* cg)
{
    if (cg->all_done && !force) return;
    const int rhs = blockIdx.x;
    __shared__ double smem[32];
    double v = 0;
    for (int k = threadIdx.x; k < ntiles; k += BLAS_BS) v += __ldcg(norm_partials + (size_t)rhs * ntiles + k);
    v = block_sum_all(v, smem);
    if (threadIdx.x == 0) cg_after_reduction(which, rhs, v, cg);
}

// x += alpha p; p = r + beta p with beta = rr_new / rr (one pass: reads x, p, r; writes x, p).  r was already
// updated by the stencil that produced q (EPI_RESID).  The last block to finish does the per-source
// bookkeeping of O5: iteration count, rr <- rr_new, the stopping test |r|/|b'| <= tol (A8), freeze flags.
// LOOP: the launch is the last kernel of the body of a WHILE graph node and decides whether another pass follows.  A
// separate instantiation, because ncu cannot profile graph kernel nodes that are able to set a conditional handle.
template <int PV, int PP, bool LOOP>
__global__ void __launch_bounds__(BLAS_BS) k_cg_update_xp(const int Vh, const int nrhs, void* __restrict__ x_, void* __restrict__ p_,
                                                          const void* __restrict__ r_, const double tol, CgScalars* cg,
                                                          const cudaGraphConditionalHandle loop)
{
    using TV = typename PT<PV>::real;
    using TP = typename PT<PP>::real;
    if (cg->all_done) {   // every source frozen: leave the device-side iteration loop, if this launch is inside one
        if constexpr (LOOP) {
            if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) cudaGraphSetConditional(loop, 0u);
        }
        return;
    }
    const int rhs = blockIdx.y;
    if (!cg->done[rhs]) {
        const TV alpha = (TV)cg->alpha[rhs];
        const TV beta = (TV)(cg->rr_new[rhs] / cg->rr[rhs]);
        char* x = (char*)x_ + field_bytes(PV, Vh, 1) * rhs;
        const char* r = (const char*)r_ + field_bytes(PV, Vh, 1) * rhs;
        char* p = (char*)p_ + field_bytes(PP, Vh, 1) * rhs;
        const int n = 3 * (int)padded_sites(Vh);
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += gridDim.x * blockDim.x) {
            const int k8 = (idx >> 5) % 3, i = (idx >> 5) / 3 * LB + (idx & 31);   // (layout block, k8, site in block)
            if (i >= Vh) continue;
            TV xv[8], rv[8];
            TP pv[8];
            load8<PV>(x, i, k8, xv);
            load8<PP>(p, i, k8, pv);
            load8<PV>(r, i, k8, rv);
#pragma unroll
            for (int k = 0; k < 8; k++) {
                xv[k] += alpha * (TV)pv[k];
                pv[k] = (TP)(rv[k] + beta * (TV)pv[k]);
            }
            store8<PV>(x, i, k8, xv);
            store8<PP>(p, i, k8, pv);
        }
    }
    if (last_block_arrive(&cg->ticket)) {
        if (threadIdx.x == 0) {
            int all = 1;
            for (int j = 0; j < nrhs; j++) {
                if (!cg->done[j]) {
                    const double v = cg->rr_new[j];
                    cg->iters[j] += 1;
                    cg->beta[j] = v / cg->rr[j];
                    cg->rr[j] = v;
                    if (tol > 0 && sqrt(v / cg->bb[j]) <= tol) cg->done[j] = 1;
                }
                all &= cg->done[j];
            }
            cg->all_done = all;
            // inside the WHILE node of a CUDA graph (api_solve.cu: cg_run): one more iteration?
            if constexpr (LOOP) {
                const int left = cg->loop_left - 1;
                cg->loop_left = left;
                cudaGraphSetConditional(loop, (!all && left > 0) ? 1u : 0u);
            }
        }
    }
}

__global__ void k_cg_loop_begin(CgScalars* cg, const int n) { cg->loop_left = n; }

inline dim3 blas_grid(const tsm_ctx* ctx, int nrhs)
{
    // the x grid does not depend on nrhs: same thread->element map and reduction tree in any batch (A14)
    long long gx = (3LL * padded_sites(ctx->g.Vh) + BLAS_BS - 1) / BLAS_BS;
    const long long cap = (long long)ctx->nsm * 4;
    if (gx > cap) gx = cap;
    return dim3((unsigned)gx, (unsigned)nrhs);
}

}  // namespace

int blas_grid_x(const tsm_ctx* ctx) { return (int)blas_grid(ctx, 1).x; }

// prec is the solve precision: F64 / F32 keep every vector in that precision; BF16 keeps
// x, r, q in fp32 and p in bf16.
#define BLAS_SWITCH(prec, CALL)                                                                   \
    switch (prec) {                                                                               \
        case TSM_F64: { constexpr int PV = TSM_F64, PP = TSM_F64; CALL; break; }                  \
        case TSM_F32: { constexpr int PV = TSM_F32, PP = TSM_F32; CALL; break; }                  \
        case TSM_BF16: { constexpr int PV = TSM_F32, PP = TSM_BF16; CALL; break; }                \
        default: return tsm_fail(ctx, TSM_EINVAL, "bad precision");                               \
    }

int launch_cg_init(tsm_ctx* ctx, int prec, int nrhs, const void* r, void* p, void* x)
{
    const dim3 grid = blas_grid(ctx, nrhs);
    if ((size_t)grid.x * nrhs > ctx->partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    BLAS_SWITCH(prec, (k_cg_init<PV, PP><<<grid, BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, nrhs, r, p, x, ctx->partials, ctx->cg)));
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_cg_reduce(tsm_ctx* ctx, int which, int nrhs, int force)
{
    if (ctx->norm_reduced) {   // k_dslash_small's last block has already summed its partials and done this step
        ctx->norm_reduced = false;
        return TSM_OK;
    }
    k_cg_reduce<<<nrhs, BLAS_BS, 0, ctx->stream>>>(which, force, ctx->norm_partials, ctx->norm_ntiles, ctx->cg);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_cg_loop_begin(tsm_ctx* ctx, int n)
{
    k_cg_loop_begin<<<1, 1, 0, ctx->stream>>>(ctx->cg, n);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_cg_update_xp(tsm_ctx* ctx, int prec, int nrhs, void* x, void* p, const void* r, double tol, unsigned long long loop, int in_loop)
{
    const dim3 grid = blas_grid(ctx, nrhs);
    const int pi = prof_begin(ctx, prec, 4, nrhs);
    if (in_loop) {
        BLAS_SWITCH(prec, (k_cg_update_xp<PV, PP, true><<<grid, BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, nrhs, x, p, r, tol, ctx->cg,
                                                                                          (cudaGraphConditionalHandle)loop)));
    } else {
        BLAS_SWITCH(prec, (k_cg_update_xp<PV, PP, false><<<grid, BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, nrhs, x, p, r, tol, ctx->cg, 0)));
    }
    prof_end(ctx, pi);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

// ------------------------------------------------------------------ N4: mixed-precision HP solver (api_solve.cu: solve_mixed)
namespace {
// Scalar bookkeeping of the fp64 defect-correction loop around the fp32 CG; one block, thread j = source j.
//   mode 0 (after the fp64 cg_init on b'): outer state <- |b'|^2, nothing done, no iterations yet
//   mode 1 (after the inner fp32 cg_init):  sources whose outer residual has converged stay frozen
//   mode 2 (after the inner solve):          iteration total += inner iterations; alpha = 1 (live) or 0 (frozen),
//                                            so that the residual stencil computes r = b' - A x for live sources
//   mode 3 (after the outer residual):       rr_outer <- |b' - A x|^2; stopping test against tol (A8)
//   mode 4 (at the end):                     copy the outer state into the fields tsm_solve reports
__global__ void k_mixed_ctl(const int mode, const int nrhs, const double tol, CgScalars* cg)
{
    const int j = threadIdx.x;
    if (j < nrhs) {
        if (mode == 0) {
            cg->bb_outer[j] = cg->bb[j];
            cg->rr_outer[j] = cg->bb[j];
            cg->iters_outer[j] = 0;
            cg->outer_done[j] = cg->done[j];
        } else if (mode == 1) {
            if (cg->outer_done[j]) cg->done[j] = 1;
        } else if (mode == 2) {
            if (!cg->outer_done[j]) cg->iters_outer[j] += cg->iters[j];
            if (!cg->outer_done[j] && cg->status[j] == TSM_EBREAKDOWN && cg->iters[j] == 0) cg->outer_done[j] = 2;   // no progress possible
            cg->alpha[j] = cg->outer_done[j] ? 0.0 : 1.0;
        } else if (mode == 3) {
            if (!cg->outer_done[j]) {
                cg->rr_outer[j] = cg->rr_new[j];
                if (sqrt(cg->rr_new[j] / cg->bb_outer[j]) <= tol) cg->outer_done[j] = 1;
            }
        } else {
            cg->iters[j] = cg->iters_outer[j];
            cg->rr[j] = cg->rr_outer[j];
            cg->bb[j] = cg->bb_outer[j];
            cg->done[j] = cg->outer_done[j] == 1;
            cg->status[j] = cg->outer_done[j] == 2 ? TSM_EBREAKDOWN : TSM_OK;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int all = 1;
        for (int k = 0; k < nrhs; k++) all &= (mode == 0 || mode == 3 || mode == 2) ? (cg->outer_done[k] != 0) : (cg->done[k] != 0);
        if (mode == 1) cg->all_done = all;                    // the inner CG's early-exit flag
        if (mode == 0 || mode == 2 || mode == 3) cg->all_outer_done = all;
    }
}

// x64 += e32 for the sources whose outer residual has not converged (fp64 accumulation of the fp32 correction)
__global__ void __launch_bounds__(BLAS_BS) k_mixed_axpy(const int Vh, void* __restrict__ x_, const void* __restrict__ e_, const CgScalars* cg)
{
    const int rhs = blockIdx.y;
    if (cg->outer_done[rhs]) return;
    char* x = (char*)x_ + field_bytes(TSM_F64, Vh, 1) * rhs;
    const char* e = (const char*)e_ + field_bytes(TSM_F32, Vh, 1) * rhs;
    const int n = 3 * (int)padded_sites(Vh);
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += gridDim.x * blockDim.x) {
        const int k8 = (idx >> 5) % 3, i = (idx >> 5) / 3 * LB + (idx & 31);
        if (i >= Vh) continue;
        double xv[8];
        float ev[8];
        load8<TSM_F64>(x, i, k8, xv);
        load8<TSM_F32>(e, i, k8, ev);
#pragma unroll
        for (int k = 0; k < 8; k++) xv[k] += (double)ev[k];
        store8<TSM_F64>(x, i, k8, xv);
    }
}
}  // namespace

int launch_mixed_ctl(tsm_ctx* ctx, int mode, int nrhs, double tol)
{
    k_mixed_ctl<<<1, 32, 0, ctx->stream>>>(mode, nrhs, tol, ctx->cg);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_mixed_axpy(tsm_ctx* ctx, int nrhs, void* x64, const void* e32)
{
    k_mixed_axpy<<<blas_grid(ctx, nrhs), BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, x64, e32, ctx->cg);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

namespace {
// |a - b|^2 per source over full-lattice fp64 native fields [parity][rhs]; one block row per source
__global__ void __launch_bounds__(BLAS_BS) k_diff_norm2(const int Vh, const int nrhs, const void* __restrict__ a,
                                                        const void* __restrict__ b, double* __restrict__ partials, CgScalars* cg)
{
    const int rhs = blockIdx.y;
    const int n = 3 * (int)padded_sites(Vh);
    double sum = 0;
    for (int par = 0; par < 2; par++) {
        const size_t off = field_bytes(TSM_F64, Vh, nrhs) * par + field_bytes(TSM_F64, Vh, 1) * rhs;
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += gridDim.x * blockDim.x) {
            const int k8 = (idx >> 5) % 3, i = (idx >> 5) / 3 * LB + (idx & 31);
            if (i >= Vh) continue;
            double u[8], v[8];
            load8<TSM_F64>((const char*)a + off, i, k8, u);
            load8<TSM_F64>((const char*)b + off, i, k8, v);
#pragma unroll
            for (int k = 0; k < 8; k++) sum += (u[k] - v[k]) * (u[k] - v[k]);
        }
    }
    __shared__ double smem[32];
    const double tot = block_sum_all(sum, smem);
    if (threadIdx.x == 0) partials[(size_t)rhs * gridDim.x + blockIdx.x] = tot;
    if (last_block_arrive(&cg->ticket)) {
        for (int j = threadIdx.x >> 5; j < nrhs; j += BLAS_BS / 32) {
            const double v = sum_partials_warp(partials, j, gridDim.x);
            if ((threadIdx.x & 31) == 0) cg->pq[j] = v;
        }
    }
}
}  // namespace

int launch_diff_norm2(tsm_ctx* ctx, int nrhs, const void* a, const void* b)
{
    const dim3 grid = blas_grid(ctx, nrhs);
    k_diff_norm2<<<grid, BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, nrhs, a, b, ctx->partials, ctx->cg);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}
