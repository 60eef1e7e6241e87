// blas.cu -- H6: the fused BLAS-1 / reduction kernels of CG on Mhat^dag Mhat (O5).
//
// Per iteration, after the four stencil launches (the last of which leaves Re<p,q> in cg->pq):
//   k_cg_update_xr : alpha = rr/pq; x += alpha p; r -= alpha q; rr' = |r|^2  (one pass, fp64 sums)
//                    last block: iteration count, stopping test |r|/|b'| <= tol (A8), beta, freeze flags
//   k_cg_update_p  : p = r + beta p
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
        for (int k = 0; k < 8; k++) { sum += (double)rv[k] * (double)rv[k]; pv[k] = (TP)rv[k]; z[k] = 0; }
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

template <int PV, int PP>
__global__ void __launch_bounds__(BLAS_BS) k_cg_update_xr(const int Vh, const int nrhs, void* __restrict__ x_, const void* __restrict__ p_,
                                                          void* __restrict__ r_, const void* __restrict__ q_, const double tol,
                                                          const double* __restrict__ norm_partials, const int ntiles,
                                                          double* __restrict__ partials, CgScalars* cg)
{
    using TV = typename PT<PV>::real;
    using TP = typename PT<PP>::real;
    if (cg->all_done) return;
    const int rhs = blockIdx.y;
    __shared__ double smem[32];
    __shared__ double pq_s;
    // Re<p,q> = |Mhat p|^2: every block sums the stencil's per-tile partials of its source in the same
    // fixed order (the partials sit in L2), so all blocks -- and any batch composition -- agree bit for bit.
    {
        double v = 0;
        for (int k = threadIdx.x; k < ntiles; k += BLAS_BS) v += __ldcg(norm_partials + (size_t)rhs * ntiles + k);
        v = block_sum_all(v, smem);
        if (threadIdx.x == 0) { pq_s = v; if (blockIdx.x == 0) cg->pq[rhs] = v; }
        __syncthreads();
    }
    const double rr = cg->rr[rhs], pq = pq_s;
    const bool frozen = cg->done[rhs] != 0;
    const bool breakdown = !(pq > 0) || !isfinite(pq) || !(rr > 0) || !isfinite(rr);   // A13
    double sum = 0;
    if (!frozen && !breakdown) {
        const TV alpha = (TV)(rr / pq);
        char* x = (char*)x_ + field_bytes(PV, Vh, 1) * rhs;
        char* r = (char*)r_ + field_bytes(PV, Vh, 1) * rhs;
        const char* q = (const char*)q_ + field_bytes(PV, Vh, 1) * rhs;
        const char* p = (const char*)p_ + field_bytes(PP, Vh, 1) * rhs;
        const int n = 3 * (int)padded_sites(Vh);
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += gridDim.x * blockDim.x) {
            const int k8 = (idx >> 5) % 3, i = (idx >> 5) / 3 * LB + (idx & 31);
            if (i >= Vh) continue;
            TV xv[8], rv[8], qv[8];
            TP pv[8];
            load8<PV>(x, i, k8, xv);
            load8<PP>(p, i, k8, pv);
            load8<PV>(r, i, k8, rv);
            load8<PV>(q, i, k8, qv);
#pragma unroll
            for (int k = 0; k < 8; k++) {
                xv[k] += alpha * (TV)pv[k];
                rv[k] -= alpha * qv[k];
                sum += (double)rv[k] * (double)rv[k];
            }
            store8<PV>(x, i, k8, xv);
            store8<PV>(r, i, k8, rv);
        }
    }
    const double tot = block_sum_all(sum, smem);
    if (threadIdx.x == 0) partials[(size_t)rhs * gridDim.x + blockIdx.x] = tot;
    if (last_block_arrive(&cg->ticket)) {
        for (int j = threadIdx.x >> 5; j < nrhs; j += BLAS_BS / 32) {
            const double v = sum_partials_warp(partials, j, gridDim.x);
            if ((threadIdx.x & 31) == 0) {
                if (!cg->done[j]) {
                    const double rr_j = cg->rr[j], pq_j = cg->pq[j];
                    if (!(pq_j > 0) || !isfinite(pq_j) || !(rr_j > 0) || !isfinite(rr_j)) {
                        cg->done[j] = 1;
                        cg->status[j] = TSM_EBREAKDOWN;
                    } else {
                        cg->iters[j] += 1;
                        cg->beta[j] = v / rr_j;
                        cg->rr[j] = v;
                        if (tol > 0 && sqrt(v / cg->bb[j]) <= tol) cg->done[j] = 1;
                    }
                }
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

template <int PV, int PP>
__global__ void __launch_bounds__(BLAS_BS) k_cg_update_p(const int Vh, void* __restrict__ p_, const void* __restrict__ r_, const CgScalars* cg)
{
    using TV = typename PT<PV>::real;
    using TP = typename PT<PP>::real;
    if (cg->all_done) return;
    const int rhs = blockIdx.y;
    if (cg->done[rhs]) return;
    const TV beta = (TV)cg->beta[rhs];
    char* p = (char*)p_ + field_bytes(PP, Vh, 1) * rhs;
    const char* r = (const char*)r_ + field_bytes(PV, Vh, 1) * rhs;
    const int n = 3 * (int)padded_sites(Vh);
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += gridDim.x * blockDim.x) {
        const int k8 = (idx >> 5) % 3, i = (idx >> 5) / 3 * LB + (idx & 31);   // (layout block, k8, site in block)
        if (i >= Vh) continue;
        TV rv[8];
        TP pv[8];
        load8<PV>(r, i, k8, rv);
        load8<PP>(p, i, k8, pv);
#pragma unroll
        for (int k = 0; k < 8; k++) pv[k] = (TP)(rv[k] + beta * (TV)pv[k]);
        store8<PP>(p, i, k8, pv);
    }
}

inline dim3 blas_grid(const tsm_ctx* ctx, int nrhs)
{
    // the x grid does not depend on nrhs: same thread->element map and reduction tree in any batch (A14)
    long long gx = (3LL * padded_sites(ctx->g.Vh) + BLAS_BS - 1) / BLAS_BS;
    const long long cap = (long long)ctx->nsm * 4;
    if (gx > cap) gx = cap;
    return dim3((unsigned)gx, (unsigned)nrhs);
}

}  // namespace

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

int launch_cg_update_xr(tsm_ctx* ctx, int prec, int nrhs, void* x, const void* p, void* r, const void* q, double tol)
{
    const dim3 grid = blas_grid(ctx, nrhs);
    if ((size_t)grid.x * nrhs > ctx->partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const int pi = prof_begin(ctx, prec, 3, nrhs);
    BLAS_SWITCH(prec, (k_cg_update_xr<PV, PP><<<grid, BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, nrhs, x, p, r, q, tol, ctx->norm_partials, ctx->norm_ntiles, ctx->partials, ctx->cg)));
    prof_end(ctx, pi);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_cg_update_p(tsm_ctx* ctx, int prec, int nrhs, void* p, const void* r)
{
    const dim3 grid = blas_grid(ctx, nrhs);
    const int pi = prof_begin(ctx, prec, 4, nrhs);
    BLAS_SWITCH(prec, (k_cg_update_p<PV, PP><<<grid, BLAS_BS, 0, ctx->stream>>>(ctx->g.Vh, p, r, ctx->cg)));
    prof_end(ctx, pi);
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
