// dslash_small.cu -- H5 for lattices that fit in L2 (hard part 4: configs 1-3): the stencil
// with the four directions of a site spread over four warps.
//
// On a 16^3 x 32 lattice a stencil launch has 65 536 output sites and takes ~10 us in k_dslash, on 4^3 x 8 (256
// sites) still ~6 us: not bandwidth (the fields sit in L2) but the CHAIN of eight dependent hop latencies per thread,
// with too few threads on the chip to hide it.  Here a CTA is 32 sites x 4 directions: warp mu loads the link pair
// and the two neighbour spinors of direction mu for its 32 sites (all loads independent: one memory latency instead
// of eight in sequence, four times as many threads in flight), forms the two hops, and leaves its 24 partial sums in
// shared memory; after one barrier warp a (= spin component a) adds the four directions' partials of its spin in a
// fixed order, applies the twist / x term / residual-update epilogue to those 3 complex numbers and stores them.
//
// The sum over directions is associated as (d0 + d1) + (d2 + d3), not sequentially as in k_dslash: a source's result
// differs from the other kernels' in rounding, so the library sends EVERY fp64 / fp32 stencil of a small-lattice
// context here (single sources and batches alike: grid = (blocks of 32 sites, sources)), and a source's result is
// still independent of its batch (A14).  Norm partials: one per (source, 32-site block), fixed trees (A19).
#include "dslash_common.cuh"
#include "reduce.cuh"

namespace {

// reals 6a .. 6a+5 (spin component a: three complex numbers) of site i
template <int PREC, bool NC> __device__ __forceinline__ void load_spin(const void* f, int i, int a, typename PT<PREC>::real* v)
{
    if constexpr (PREC == TSM_F64) {
        const char* p = site_ptr<12>(f, i) + (3 * a) * LB_ROW;
#pragma unroll
        for (int c = 0; c < 3; c++) { const double2 w = ld16<NC, double2>(p + c * LB_ROW); v[2 * c] = w.x; v[2 * c + 1] = w.y; }
    } else {
        const char* p = site_ptr<6>(f, i);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int r = 6 * a + 2 * c;   // even: an 8-byte piece of chunk r / 4
            const char* q = p + (r >> 2) * LB_ROW + (r & 3) * 4;
            float2 w;
            if constexpr (NC) w = __ldg(reinterpret_cast<const float2*>(q));
            else w = *reinterpret_cast<const float2*>(q);
            v[2 * c] = w.x; v[2 * c + 1] = w.y;
        }
    }
}
template <int PREC> __device__ __forceinline__ void store_spin(void* f, int i, int a, const typename PT<PREC>::real* v)
{
    if constexpr (PREC == TSM_F64) {
        char* p = site_ptr<12>(f, i) + (3 * a) * LB_ROW;
#pragma unroll
        for (int c = 0; c < 3; c++) *reinterpret_cast<double2*>(p + c * LB_ROW) = make_double2(v[2 * c], v[2 * c + 1]);
    } else {
        char* p = site_ptr<6>(f, i);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int r = 6 * a + 2 * c;
            *reinterpret_cast<float2*>(p + (r >> 2) * LB_ROW + (r & 3) * 4) = make_float2(v[2 * c], v[2 * c + 1]);
        }
    }
}

// both hops of direction MU of site i into part[24] (zero on entry)
template <int PREC, int RECON, bool DAGGER, int MU, bool NC>
__device__ __forceinline__ void two_hops(const void* pack, const char* in, int i, int nf, int nbk, typename PT<PREC>::real ph_f,
                                         typename PT<PREC>::real ph_b, typename PT<PREC>::real* part)
{
    using T = typename PT<PREC>::real;
    constexpr int SF = DAGGER ? +1 : -1;   // forward hop carries (1 - g_mu), dagger swaps
    T uf[18], ub[18], pf[24], pb[24], h[12], gq[12];
    load_link_pair<PREC, RECON>(pack, i, MU, uf, ub);
    load_spinor<PREC, NC>(in, nf, pf);
    load_spinor<PREC, NC>(in, nbk, pb);
    project<T, MU, SF>(pf, h);
    if (MU == 3 && ph_f != 1) {   // time-boundary phase (A22)
#pragma unroll
        for (int k = 0; k < 12; k++) h[k] *= ph_f;
    }
    su3_mul(uf, h, gq);
    su3_mul(uf, h + 6, gq + 6);
    accumulate<T, MU, SF>(gq, part);
    project<T, MU, -SF>(pb, h);
    if (MU == 3 && ph_b != 1) {
#pragma unroll
        for (int k = 0; k < 12; k++) h[k] *= ph_b;
    }
    su3_mul(ub, h, gq);
    su3_mul(ub, h + 6, gq + 6);
    accumulate<T, MU, -SF>(gq, part);
}

// One 32-site layout block `blk` of one source: four warps = four directions, then four warps = four spin components.
// in / xf / out point at that source's fields; sm, red: the CTA's exchange buffers (the caller puts a barrier between two
// calls).  Returns, in thread 0, the block's contribution to the fused norm.  NC: gather through ld.global.nc (false inside
// the persistent CG kernel, where the gathered field is rewritten between two phases of the same launch).  Shared by
// k_dslash_small and k_cg_persistent_small, so that the two give a source bit-identical results.
template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI, bool NC>
__device__ __forceinline__ double small_block(const Geom& g, const int par, const int blk, const void* pack, const char* in, const char* xf,
                                              char* out, const DslashCoef& cf, const typename PT<PREC>::real alpha,
                                              typename PT<PREC>::real (*sm)[24][32], double* red)
{
    using T = typename PT<PREC>::real;
    const int Vh = g.Vh;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;   // w: direction in the first half, spin component in the second
    const int i = blk * LB + lane;
    const bool live = i < Vh;
    // the own-site x and r vectors of the second half (spin component w) are requested BEFORE the hops: their latency then
    // overlaps the gathers instead of following the barrier (the same values: nothing writes them in between)
    T xv[6] = {}, rv[6] = {};
    if (XPAY && live) load_spin<PREC, NC>(xf, i, w, xv);
    if (EPI == EPI_RESID && live) load_spin<PREC, false>(out, i, w, rv);
    {
        T part[24];
#pragma unroll
        for (int k = 0; k < 24; k++) part[k] = 0;
        if (live) {
            const SiteCoord s = decode_site(g, i, par);
            int nb[8];
            neighbours(g, i, s, nb);
            const T ph_f = (s.t == g.L[3] - 1) ? (T)g.theta : (T)1, ph_b = (s.t == 0) ? (T)g.theta : (T)1;
            switch (w) {   // warp-uniform
                case 0: two_hops<PREC, RECON, DAGGER, 0, NC>(pack, in, i, nb[0], nb[1], ph_f, ph_b, part); break;
                case 1: two_hops<PREC, RECON, DAGGER, 1, NC>(pack, in, i, nb[2], nb[3], ph_f, ph_b, part); break;
                case 2: two_hops<PREC, RECON, DAGGER, 2, NC>(pack, in, i, nb[4], nb[5], ph_f, ph_b, part); break;
                default: two_hops<PREC, RECON, DAGGER, 3, NC>(pack, in, i, nb[6], nb[7], ph_f, ph_b, part); break;
            }
        }
#pragma unroll
        for (int k = 0; k < 24; k++) sm[w][k][lane] = part[k];
    }
    __syncthreads();
    // second half: warp w finishes spin component w of the 32 sites
    const int a = w;
    double nrm = 0.0;
    if (live) {
        T v[6], o[6];
#pragma unroll
        for (int c = 0; c < 6; c++) v[c] = (sm[0][6 * a + c][lane] + sm[1][6 * a + c][lane]) + (sm[2][6 * a + c][lane] + sm[3][6 * a + c][lane]);
        const T cdr = (T)(a < 2 ? cf.d.up_re : cf.d.lo_re), cdi = (T)(a < 2 ? cf.d.up_im : cf.d.lo_im);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            // explicit chains: k_dslash_small and k_cg_persistent_small must round alike, so which of two products is
            // fused is not left to the compiler
            o[2 * c] = fma_(cdr, v[2 * c], -(cdi * v[2 * c + 1]));
            o[2 * c + 1] = fma_(cdr, v[2 * c + 1], cdi * v[2 * c]);
        }
        if (XPAY) {
            const T cxr = (T)(a < 2 ? cf.x.up_re : cf.x.lo_re), cxi = (T)(a < 2 ? cf.x.up_im : cf.x.lo_im);
#pragma unroll
            for (int c = 0; c < 3; c++) {
                o[2 * c] = fma_(cxr, xv[2 * c], fma_(-cxi, xv[2 * c + 1], o[2 * c]));
                o[2 * c + 1] = fma_(cxr, xv[2 * c + 1], fma_(cxi, xv[2 * c], o[2 * c + 1]));
            }
        }
        if (EPI == EPI_RESID) {   // out is the CG residual r (same precision as the spinors here): r -= alpha q
#pragma unroll
            for (int c = 0; c < 6; c++) { rv[c] = fma_(-alpha, o[c], rv[c]); nrm = fma((double)rv[c], (double)rv[c], nrm); }
            store_spin<PREC>(out, i, a, rv);
        } else {
            store_spin<PREC>(out, i, a, o);
            if (EPI == EPI_NORM) {
#pragma unroll
                for (int c = 0; c < 6; c++) nrm = fma((double)o[c], (double)o[c], nrm);
            }
        }
    }
    double tot = 0.0;
    if (EPI != EPI_NONE) {
        const double ws = warp_sum(nrm);
        if (lane == 0) red[w] = ws;
        __syncthreads();
        if (threadIdx.x == 0) tot = (red[0] + red[1]) + (red[2] + red[3]);
    }
    return tot;
}

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI>
__global__ void __launch_bounds__(128) k_dslash_small(const Geom g, const int par, const void* __restrict__ pack, const void* __restrict__ in_,
                                                      const void* __restrict__ x_, void* out_, const DslashCoef cf,
                                                      double* __restrict__ partials, CgScalars* __restrict__ cg, const int check_done)
{
    using T = typename PT<PREC>::real;
    __shared__ T sm[4][24][32];
    __shared__ double red[4];
    if (check_done && cg->all_done) return;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int rhs = blockIdx.y;
    const size_t fb = field_bytes(PREC, g.Vh, 1);
    T alpha = 0;
    if (EPI == EPI_RESID) alpha = (T)cg->alpha[rhs];
    const double tot = small_block<PREC, RECON, DAGGER, XPAY, EPI, true>(g, par, blockIdx.x, pack, (const char*)in_ + fb * rhs, (const char*)x_ + fb * rhs,
                                                                         (char*)out_ + fb * rhs, cf, alpha, sm, red);
    if (EPI != EPI_NONE) {
        if (threadIdx.x == 0) partials[(size_t)rhs * gridDim.x + blockIdx.x] = tot;
        // The last block of the grid to finish sums every source's partials (one warp per source, an order that
        // depends on the number of blocks only) and does what k_cg_reduce would: on these lattices a separate
        // reduction launch costs as much as the stencil itself.
        if (last_block_arrive(&cg->ticket)) {
            for (int j = w; j < (int)gridDim.y; j += 4) {
                const double v = sum_partials_warp(partials, j, gridDim.x);
                if (lane == 0) cg_after_reduction(EPI == EPI_RESID ? 1 : 0, j, v, cg);
            }
        }
    }
}

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI>
int launch_small_t(tsm_ctx* ctx, int par, int nrhs, const void* pack, const void* in, const void* x, void* out, const DslashCoef& c,
                   int check_done)
{
    const int nblocks = (int)(padded_sites(ctx->g.Vh) / LB);
    if (EPI != EPI_NONE && (size_t)nblocks * nrhs > ctx->norm_partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const int pi = prof_begin(ctx, PREC, EPI == EPI_RESID ? 3 : (EPI == EPI_NORM ? 2 : (XPAY ? 1 : 0)), nrhs);
    k_dslash_small<PREC, RECON, DAGGER, XPAY, EPI><<<dim3(nblocks, nrhs), 128, 0, ctx->stream>>>(ctx->g, par, pack, in, x, out, c, ctx->norm_partials,
                                                                                                   ctx->cg, check_done);
    prof_end(ctx, pi);
    ctx->launches++;
    ctx->norm_ntiles = nblocks;
    ctx->norm_reduced = EPI != EPI_NONE;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

template <int PREC, int RECON>
int launch_small_p(tsm_ctx* ctx, int par, bool dagger, int nrhs, const void* pack, const void* in, const void* x, void* out,
                   const DslashCoef& c, int epi, int check_done)
{
    const bool xpay = x != nullptr;
#define GO(DG, XP, EP) return launch_small_t<PREC, RECON, DG, XP, EP>(ctx, par, nrhs, pack, in, x, out, c, check_done)
    if (!dagger && !xpay && epi == EPI_NONE) GO(false, false, EPI_NONE);
    if (!dagger && xpay && epi == EPI_NONE) GO(false, true, EPI_NONE);
    if (dagger && !xpay && epi == EPI_NONE) GO(true, false, EPI_NONE);
    if (dagger && xpay && epi == EPI_NONE) GO(true, true, EPI_NONE);
    if (!dagger && xpay && epi == EPI_NORM) GO(false, true, EPI_NORM);
    if (dagger && xpay && epi == EPI_RESID) GO(true, true, EPI_RESID);
#undef GO
    return tsm_fail(ctx, TSM_EINVAL, "unsupported dslash variant");
}

}  // namespace

// fp64 / fp32, any nrhs >= 1.  mode bits as in launch_dslash.
int launch_dslash_small(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x, void* out,
                        const DslashCoef& c, int mode)
{
    const int chk = (mode >> 1) & 1, nm = (mode & 4) ? EPI_RESID : ((mode & 1) ? EPI_NORM : EPI_NONE);
    if (prec == TSM_F64) return launch_small_p<TSM_F64, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge64[out_parity], in, x, out, c, nm, chk);
    if (prec == TSM_F32) {
        if (ctx->recon == 18) return launch_small_p<TSM_F32, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, nm, chk);
        return launch_small_p<TSM_F32, 12>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, nm, chk);
    }
    return tsm_fail(ctx, TSM_EINVAL, "small-lattice stencil: unsupported precision");
}

// ------------------------------------------------------------------ the persistent CG kernel in this file's formulation
// k_cg_persistent (dslash.cu) with small_block() as the stencil: one cooperative launch for the whole iteration loop of O5
// on the lattices where k_dslash_small is the stencil (a phase is then two dependent gathers per thread instead of eight).
// Same partials per 32-site block, same order over blocks (sum_partials_warp), same update formula as k_cg_update_xp: a
// source's iterate is bit-identical to the kernel-by-kernel path with k_dslash_small.
#include <cooperative_groups.h>

namespace {

namespace cgp = cooperative_groups;

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI>
__device__ __forceinline__ void pcgs_stencil(const PcgArgs& a, const int par, const void* in_, const void* x_, void* out_, const DslashCoef& cf,
                                             const double* s_alpha, double* partials, typename PT<PREC>::real (*sm)[24][32], double* red)
{
    using T = typename PT<PREC>::real;
    const size_t fb = field_bytes(PREC, a.g.Vh, 1);
    for (int blk = blockIdx.x; blk < a.ntiles; blk += gridDim.x)
        for (int rhs = 0; rhs < a.nrhs; rhs++) {
            T alpha = 0;
            if (EPI == EPI_RESID) alpha = (T)s_alpha[rhs];
            const double tot = small_block<PREC, RECON, DAGGER, XPAY, EPI, false>(a.g, par, blk, a.pack[par], (const char*)in_ + fb * rhs,
                                                                                  (const char*)x_ + fb * rhs, (char*)out_ + fb * rhs, cf, alpha, sm, red);
            if (EPI != EPI_NONE && threadIdx.x == 0) partials[(size_t)rhs * a.ntiles + blk] = tot;
            __syncthreads();   // sm and red are reused by the next (block, source)
        }
}

template <int PREC, int RECON>
__global__ void __launch_bounds__(128) k_cg_persistent_small(const PcgArgs a)
{
    using T = typename PT<PREC>::real;
    cgp::grid_group grid = cgp::this_grid();
    __shared__ T sm[4][24][32];
    __shared__ double red[4];
    __shared__ double s_alpha[TSM_MAX_NRHS], s_rr[TSM_MAX_NRHS], s_rrnew[TSM_MAX_NRHS], s_beta[TSM_MAX_NRHS], s_pq[TSM_MAX_NRHS];
    __shared__ double s_bb[TSM_MAX_NRHS];
    __shared__ int s_done[TSM_MAX_NRHS], s_iters[TSM_MAX_NRHS], s_status[TSM_MAX_NRHS];
    __shared__ int s_all, s_broke;
    CgScalars* cg = a.cg;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int Vh = a.g.Vh, nrhs = a.nrhs;
    const size_t fb = field_bytes(PREC, Vh, 1);
    if (tid < nrhs) {
        s_rr[tid] = cg->rr[tid]; s_done[tid] = cg->done[tid]; s_iters[tid] = cg->iters[tid]; s_status[tid] = cg->status[tid];
        s_beta[tid] = cg->beta[tid]; s_pq[tid] = cg->pq[tid]; s_alpha[tid] = 0.0; s_rrnew[tid] = cg->rr_new[tid];
        s_bb[tid] = cg->bb[tid];
    }
    if (tid == 0) { s_all = cg->all_done; s_broke = 0; }
    __syncthreads();
    double* part_w = a.partials;
    double* part_r = a.partials + (size_t)nrhs * a.ntiles;

    if (a.whole) {
        // ---- H4 (tsm_solve): aux = R^-1 eta_o; bhat = eta_e + kappa D_eo aux (into w); t = Rb^-1 D_oe^dag bhat; b' = Mhat^dag bhat (into r)
        if (tid < 96) {   // 32 sites x 3 groups of 8 reals, k_twist's arithmetic
            const int k8 = tid >> 5;
            for (int rhs = 0; rhs < nrhs; rhs++)
                for (int blk = blockIdx.x; blk < a.ntiles; blk += gridDim.x) {
                    const int i = blk * LB + lane;
                    if (i >= Vh) continue;
                    T v[8], o[8];
                    load8<PREC, false>((const char*)a.s_o + fb * rhs, i, k8, v);
                    twist8<T>(a.tw_rinv, k8, v, o);
                    store8<PREC>((char*)a.aux + fb * rhs, i, k8, o);
                }
        }
        grid.sync();
        pcgs_stencil<PREC, RECON, false, true, EPI_NONE>(a, 0, a.aux, a.x, a.w, a.cp1, s_alpha, nullptr, sm, red);
        grid.sync();
        pcgs_stencil<PREC, RECON, true, false, EPI_NONE>(a, 1, a.w, nullptr, a.t, a.cp2, s_alpha, nullptr, sm, red);
        grid.sync();
        pcgs_stencil<PREC, RECON, true, true, EPI_NONE>(a, 0, a.t, a.w, a.r, a.cp3, s_alpha, nullptr, sm, red);
        // ---- O5 start (k_cg_init): x0 = 0, p0 = r0 = b', |b'|^2.  Own blocks only (this CTA's warps have just written them and
        // pcgs_stencil ends on a block barrier).  |r|^2 is left per (block, group of 8 reals) = per warp of k_cg_init ...
        if (tid < 96) {
            const int k8 = tid >> 5;
            for (int rhs = 0; rhs < nrhs; rhs++)
                for (int blk = blockIdx.x; blk < a.ntiles; blk += gridDim.x) {
                    const int i = blk * LB + lane;
                    double sum = 0;
                    if (i < Vh) {
                        T rv[8], z[8];
                        load8<PREC, false>((const char*)a.r + fb * rhs, i, k8, rv);
#pragma unroll
                        for (int k = 0; k < 8; k++) { sum = fma((double)rv[k], (double)rv[k], sum); z[k] = 0; }   // k_cg_init's chain, not left to contraction
                        store8<PREC>((char*)a.p + fb * rhs, i, k8, rv);
                        store8<PREC>((char*)a.x + fb * rhs, i, k8, z);
                    }
                    const double gsum = warp_sum(sum);
                    if (lane == 0) a.init_groups[(size_t)rhs * 3 * a.ntiles + 3 * blk + k8] = gsum;
                }
        }
        grid.sync();
        // ... and summed in k_cg_init's order: its block b adds its 8 warps (groups 8b .. 8b+7) serially, then one warp adds
        // the blocks lane-strided and by the shuffle tree (sum_partials_warp)
        for (int j = wid; j < nrhs; j += 4) {
            const double* gr = a.init_groups + (size_t)j * 3 * a.ntiles;
            const int ng = 3 * a.ntiles;
            double v = 0;
            for (int b = lane; b < a.init_gx; b += 32) {
                double pb = 0;
                for (int k = 0; k < 8; k++) pb += (8 * b + k < ng) ? __ldcg(gr + 8 * b + k) : 0.0;
                v += pb;
            }
            v = warp_sum(v);
            if (lane == 0) {
                s_rr[j] = v; s_bb[j] = v; s_pq[j] = 0; s_beta[j] = 0; s_iters[j] = 0; s_status[j] = TSM_OK; s_done[j] = !(v > 0);
                s_alpha[j] = 0.0;
            }
        }
        __syncthreads();
        if (tid == 0) {
            int all = 1;
            for (int j = 0; j < nrhs; j++) all &= s_done[j];
            s_all = all;
        }
        __syncthreads();
    }

    for (int it = 0; it < a.max_iter && !s_all; it++) {
        pcgs_stencil<PREC, RECON, false, false, EPI_NONE>(a, 1, a.p, nullptr, a.t, a.c1, s_alpha, nullptr, sm, red);   // t = R^-1 D_oe p
        grid.sync();
        pcgs_stencil<PREC, RECON, false, true, EPI_NORM>(a, 0, a.t, a.p, a.w, a.c2, s_alpha, part_w, sm, red);         // w = Mhat p; |w|^2
        grid.sync();
        for (int j = wid; j < nrhs; j += 4) {   // alpha = rr / |w|^2 (cg_after_reduction, which == 0)
            const double v = sum_partials_warp(part_w, j, a.ntiles);
            if (lane == 0) {
                s_pq[j] = v;
                double alpha = 0.0;
                if (!s_done[j]) {
                    const double rr = s_rr[j];
                    if (!(v > 0) || !isfinite(v) || !(rr > 0) || !isfinite(rr)) { s_done[j] = 1; s_status[j] = TSM_EBREAKDOWN; s_broke = 1; }
                    else alpha = rr / v;
                }
                s_alpha[j] = alpha;
            }
        }
        __syncthreads();
        pcgs_stencil<PREC, RECON, true, false, EPI_NONE>(a, 1, a.w, nullptr, a.t, a.c3, s_alpha, nullptr, sm, red);    // t = Rb^-1 D_oe^dag w
        grid.sync();
        pcgs_stencil<PREC, RECON, true, true, EPI_RESID>(a, 0, a.t, a.w, a.r, a.c4, s_alpha, part_r, sm, red);         // r -= alpha Mhat^dag w; |r|^2
        grid.sync();
        for (int j = wid; j < nrhs; j += 4) {   // rr' (which == 1)
            const double v = sum_partials_warp(part_r, j, a.ntiles);
            if (lane == 0) s_rrnew[j] = v;
        }
        __syncthreads();
        // x += alpha p; p = r + beta p on this CTA's own blocks: 96 threads = 32 sites x 3 groups of 8 reals
        if (tid < 96) {
            const int k8 = tid >> 5;
            for (int rhs = 0; rhs < nrhs; rhs++) {
                if (s_done[rhs]) continue;
                const T alpha = (T)s_alpha[rhs];
                const T beta = (T)(s_rrnew[rhs] / s_rr[rhs]);
                char* x = (char*)a.x + fb * rhs;
                char* p = (char*)a.p + fb * rhs;
                const char* r = (const char*)a.r + fb * rhs;
                for (int blk = blockIdx.x; blk < a.ntiles; blk += gridDim.x) {
                    const int i = blk * LB + lane;
                    if (i >= Vh) continue;
                    T xv[8], pv[8], rv[8];
                    load8<PREC, false>(x, i, k8, xv);
                    load8<PREC, false>(p, i, k8, pv);
                    load8<PREC, false>(r, i, k8, rv);
#pragma unroll
                    for (int k = 0; k < 8; k++) {
                        xv[k] += alpha * pv[k];
                        pv[k] = rv[k] + beta * pv[k];
                    }
                    store8<PREC>(x, i, k8, xv);
                    store8<PREC>(p, i, k8, pv);
                }
            }
        }
        __syncthreads();
        if (tid == 0) {   // the bookkeeping of k_cg_update_xp's last block
            int all = 1;
            for (int j = 0; j < nrhs; j++) {
                if (!s_done[j]) {
                    const double v = s_rrnew[j];
                    s_iters[j] += 1;
                    s_beta[j] = v / s_rr[j];
                    s_rr[j] = v;
                    if (a.tol > 0 && sqrt(v / s_bb[j]) <= a.tol) s_done[j] = 1;
                }
                all &= s_done[j];
            }
            s_all = all;
        }
        grid.sync();
    }
    // ---- H7: s_o = R^-1 (eta_o + kappa D_oe x), in place (a thread reads and rewrites only its own components)
    if (a.whole) pcgs_stencil<PREC, RECON, false, true, EPI_NONE>(a, 1, a.x, a.s_o, a.s_o, a.crec, s_alpha, nullptr, sm, red);
    if (blockIdx.x == 0) {
        __syncthreads();
        if (tid < nrhs) {
            cg->bb[tid] = s_bb[tid];
            cg->rr[tid] = s_rr[tid]; cg->done[tid] = s_done[tid]; cg->iters[tid] = s_iters[tid]; cg->status[tid] = s_status[tid];
            cg->beta[tid] = s_beta[tid]; cg->pq[tid] = s_pq[tid]; cg->alpha[tid] = s_alpha[tid]; cg->rr_new[tid] = s_rrnew[tid];
        }
        if (tid == 0) {
            cg->all_done = s_all;
            if (s_broke) cg->sticky_breakdown = 1;
        }
    }
}

template <int PREC, int RECON> int launch_pcgs_t(tsm_ctx* ctx, PcgArgs& a)
{
    auto kern = k_cg_persistent_small<PREC, RECON>;
    static int resident[64] = {0};
    if (ctx->device >= 64) return tsm_fail(ctx, TSM_EINVAL, "persistent CG: device index beyond 63");
    if (!resident[ctx->device]) {
        int nb = 0;
        TSM_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 128, 0));
        if (nb < 1) return tsm_fail(ctx, TSM_ECUDA, "persistent CG kernel does not fit an SM");
        resident[ctx->device] = nb;
    }
    int grid = ctx->nsm * resident[ctx->device];
    if (grid > a.ntiles) grid = a.ntiles;
    void* params[] = {(void*)&a};
    TSM_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(128), params, 0, ctx->stream));
    ctx->launches++;
    return TSM_OK;
}

}  // namespace

int launch_cg_persistent_small(tsm_ctx* ctx, int prec, PcgArgs& a)
{
    if (prec == TSM_F64) return launch_pcgs_t<TSM_F64, 18>(ctx, a);
    if (ctx->recon == 18) return launch_pcgs_t<TSM_F32, 18>(ctx, a);
    return launch_pcgs_t<TSM_F32, 12>(ctx, a);
}
