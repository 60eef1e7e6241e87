// dslash_tile.cu -- H5 for batches of sources (fp32 and bf16 storage): the stencil of dslash.cu with
// the links of a tile staged in shared memory by bulk asynchronous copies (TMA, cp.async.bulk).
//
// A persistent CTA owns one tile of 128 output sites at a time and applies the stencil to ALL
// sources of the batch before it moves on.  The 8 links of the tile's sites are one contiguous
// piece of the link pack (4 layout blocks x NCH chunks x 512 B = 72 KB with 18 reals, 48 KB with
// 12): a single cp.async.bulk brings it into shared memory, completion is signalled on an
// mbarrier, and the copy for the CTA's NEXT tile is issued before the current tile is computed
// (two buffers), so the only loads that come straight from DRAM are never waited for by the
// arithmetic.  Every link is then read from HBM/L2 once per tile whatever the batch size, and
// R sources are handled per thread with the link pair held in registers (R x fewer shared-memory
// reads, R independent dependency chains).  blockDim = (128 sites, RY source rows); a CTA loops over
// G = ceil(nrhs / (RY * R)) groups of sources.  Neighbour spinors come through L1/L2 (ld.global.nc).
// Shapes in use (measured at 32^3 x 64, 12 sources, inside the CG): the plain launches
// (no x term, no epilogue) run 3 rows x 2 sources per thread (168 registers, 12 warps: 821 us against 882 us
// for 4 x 1); the launches with an x term or an epilogue run 3 rows x 1 source (168 registers, 12 warps) and request
// the own-site x / r vectors BEFORE the hops, so that those first-touch DRAM streams are in flight during the
// gathers (S2 1039 -> 978 us, S4 1112 -> 1047 us against 4 rows x 1 source with the loads in the epilogue; with two
// sources per thread they were 1113-1243 us: the second source's x / r vectors do not fit beside the accumulators).
// Batches whose size is not a multiple of 3 keep 4 rows x 1 source (plain launches of 4 sources: 2 rows x 2).
//
// Arithmetic per source is the same sequence of operations as in dslash.cu (same projection,
// same FMA chains, same accumulation order over mu), so a source's result does not depend on the
// batch it is in (reading A14).
#include <cstdlib>

#include "bulk_copy.cuh"
#include "dslash_common.cuh"
#include "reduce.cuh"

namespace {

constexpr int TT = 128;   // sites per tile = blockDim.x = 4 layout blocks

// both links of direction MU of the thread's site from the staged tile (same layout as the pack)
template <int RECON, int MU> __device__ __forceinline__ void lds_link_pair(const char* tile_links, int tx, float* uf, float* ub)
{
    constexpr int NCH = RECON == 18 ? 36 : 24;
    const char* p = tile_links + (tx >> 5) * (NCH * LB_ROW) + (tx & 31) * 16;
    if constexpr (RECON == 18) {
        float l[36];
#pragma unroll
        for (int j = 0; j < 9; j++) {
            const float4 v = *reinterpret_cast<const float4*>(p + (9 * MU + j) * LB_ROW);
            l[4 * j] = v.x; l[4 * j + 1] = v.y; l[4 * j + 2] = v.z; l[4 * j + 3] = v.w;
        }
#pragma unroll
        for (int j = 0; j < 18; j++) { uf[j] = l[j]; ub[j] = l[18 + j]; }
    } else {
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const float4 v = *reinterpret_cast<const float4*>(p + (6 * MU + j) * LB_ROW);
            uf[4 * j] = v.x; uf[4 * j + 1] = v.y; uf[4 * j + 2] = v.z; uf[4 * j + 3] = v.w;
        }
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const float4 v = *reinterpret_cast<const float4*>(p + (6 * MU + 3 + j) * LB_ROW);
            ub[4 * j] = v.x; ub[4 * j + 1] = v.y; ub[4 * j + 2] = v.z; ub[4 * j + 3] = v.w;
        }
        reconstruct_row2(uf);
        reconstruct_row2(ub);
    }
}

// one direction, R sources: links once, then the forward and the backward hop of every source
template <int PREC, int RECON, bool DAGGER, int MU, int R>
__device__ __forceinline__ void hop_direction_r(const char* tile_links, int tx, const char* in, size_t fb, const int* nb, float ph_f,
                                                float ph_b, float (*acc)[24])
{
    constexpr int SF = DAGGER ? +1 : -1;   // forward hop carries (1 - g_mu), dagger swaps
    float uf[18], ub[18];
    lds_link_pair<RECON, MU>(tile_links, tx, uf, ub);
#pragma unroll
    for (int r = 0; r < R; r++) {
        float psi[24], h[12], gq[12];
        load_spinor<PREC>(in + fb * r, nb[2 * MU], psi);
        project<float, MU, SF>(psi, h);
        if (MU == 3 && ph_f != 1) rscale_f32<6>(ph_f, h);   // time-boundary phase (A22); skipping a multiplication by one is exact
        su3_mul(uf, h, gq);
        su3_mul(uf, h + 6, gq + 6);
        accumulate<float, MU, SF>(gq, acc[r]);
    }
#pragma unroll
    for (int r = 0; r < R; r++) {
        float psi[24], h[12], gq[12];
        load_spinor<PREC>(in + fb * r, nb[2 * MU + 1], psi);
        project<float, MU, -SF>(psi, h);
        if (MU == 3 && ph_b != 1) rscale_f32<6>(ph_b, h);
        su3_mul(ub, h, gq);
        su3_mul(ub, h + 6, gq + 6);
        accumulate<float, MU, -SF>(gq, acc[r]);
    }
}

// cb index of the first site of tile `tile`.  With slab traversal (S a multiple of 128) the tiles
// follow the z-slab / t order of dslash.cu's traverse_site; otherwise plain cb order.  Either way a
// tile is 128 consecutive cb sites starting at a multiple of 128 (4 whole layout blocks).
__device__ __forceinline__ int tile_base(const Geom& g, int tile, int slab)
{
    const int v0 = tile * TT;
    if (!slab) return v0;
    unsigned q1, r, zb, t, zi, rest;
    g.dSB.divmod((unsigned)v0, q1, r);
    g.dLt.divmod(q1, zb, t);
    g.dS.divmod(r, zi, rest);
    return (int)(t * g.Vsh + (zb * g.bz + zi) * g.S + rest);
}

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI, int RY, int R>
__global__ void __launch_bounds__(TT * RY, 1)
k_dslash_tile(const Geom g, const int par, const int nrhs, const int ntiles, const int slab, const void* __restrict__ pack,
              const void* __restrict__ in_, const void* __restrict__ x_, void* out_, const DslashCoef cf,
              double* __restrict__ partials, CgScalars* __restrict__ cg, const int check_done, const int fuse_reduce)
{
    constexpr int NCH = RECON == 18 ? 36 : 24;
    constexpr unsigned TILE_BYTES = 4 * NCH * LB_ROW;
    extern __shared__ __align__(128) char smem[];
    __shared__ __align__(8) uint64_t bar[2];
    constexpr int PR = PREC == TSM_BF16 ? TSM_F32 : PREC;   // storage of the CG residual (EPI_RESID)
    __shared__ double red[EPI != EPI_NONE ? RY * 2 * 4 * R : 1];
    if (check_done && cg->all_done) return;
    const int Vh = g.Vh;
    const int nblocks = (int)(padded_sites(Vh) / LB);
    const size_t fb = field_bytes(PREC, Vh, 1), fbo = field_bytes(EPI == EPI_RESID ? PR : PREC, Vh, 1);
    const float cxur = (float)cf.x.up_re, cxui = (float)cf.x.up_im, cxlr = (float)cf.x.lo_re, cxli = (float)cf.x.lo_im;
    const float cdur = (float)cf.d.up_re, cdui = (float)cf.d.up_im, cdlr = (float)cf.d.lo_re, cdli = (float)cf.d.lo_im;
    const bool d_real = cdui == 0.f && cdli == 0.f;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const bool leader = (tx == 0 && ty == 0);

    auto issue = [&](int tile, int b) {
        const int i0 = tile_base(g, tile, slab);
        int nb_ = nblocks - (i0 >> 5);
        if (nb_ > 4) nb_ = 4;
        const unsigned bytes = (unsigned)nb_ * NCH * LB_ROW;
        mbar_expect_tx(&bar[b], bytes);
        bulk_g2s(smem + (size_t)b * TILE_BYTES, (const char*)pack + (size_t)(i0 >> 5) * (NCH * LB_ROW), bytes, &bar[b]);
    };

    if (leader) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (leader && (int)blockIdx.x < ntiles) issue(blockIdx.x, 0);

    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, it++) {
        const int b = it & 1;
        // buffer b^1 was last read in iteration it-1, which ended with __syncthreads()
        if (leader && tile + (int)gridDim.x < ntiles) issue(tile + gridDim.x, b ^ 1);
        const int i = tile_base(g, tile, slab) + tx;
        const bool live = i < Vh;
        SiteCoord s = decode_site(g, live ? i : 0, par);
        int nb[8];
        neighbours(g, live ? i : 0, s, nb);
        const float ph_f = (s.t == g.L[3] - 1) ? (float)g.theta : 1.f;
        const float ph_b = (s.t == 0) ? (float)g.theta : 1.f;
        mbar_wait(&bar[b], (unsigned)((it >> 1) & 1));
        const char* links = smem + (size_t)b * TILE_BYTES;

        for (int grp = 0; grp * RY * R < nrhs; grp++) {
            const int rhs0 = (grp * RY + ty) * R;
            const bool act = live && rhs0 < nrhs;      // R divides nrhs: a row is wholly inside or outside
            double nrm[R];
#pragma unroll
            for (int r = 0; r < R; r++) nrm[r] = 0.0;
            if (act) {
                const char* in = (const char*)in_ + fb * rhs0;
                float acc[R][24];
#pragma unroll
                for (int r = 0; r < R; r++)
#pragma unroll
                    for (int k = 0; k < 24; k++) acc[r][k] = 0.f;
                // 3 rows x 1 source: the registers that 12 warps leave free hold the epilogue's own-site inputs, requested
                // now (EARLY); otherwise they are loaded where they are used
                constexpr bool EARLY = RY == 3 && R == 1 && (XPAY || EPI == EPI_RESID);
                float xe[EARLY && XPAY ? 24 : 1], rve[EARLY && EPI == EPI_RESID ? 24 : 1];
                if constexpr (EARLY && XPAY) load_spinor<PREC>((const char*)x_ + fb * rhs0, i, xe);
                if constexpr (EARLY && EPI == EPI_RESID) load_spinor<PR, false>((const char*)out_ + fbo * rhs0, i, rve);   // coherent: r is rewritten below
                hop_direction_r<PREC, RECON, DAGGER, 0, R>(links, tx, in, fb, nb, ph_f, ph_b, acc);
                hop_direction_r<PREC, RECON, DAGGER, 1, R>(links, tx, in, fb, nb, ph_f, ph_b, acc);
                hop_direction_r<PREC, RECON, DAGGER, 2, R>(links, tx, in, fb, nb, ph_f, ph_b, acc);
                hop_direction_r<PREC, RECON, DAGGER, 3, R>(links, tx, in, fb, nb, ph_f, ph_b, acc);
#pragma unroll
                for (int r = 0; r < R; r++) {
                    float o[24];
                    if (d_real) { cscale_real_f32<6>(cdur, acc[r], o); cscale_real_f32<6>(cdlr, acc[r] + 12, o + 12); }   // Td real (-kappa^2)
                    else { cscale_f32<6>(cdur, cdui, acc[r], o); cscale_f32<6>(cdlr, cdli, acc[r] + 12, o + 12); }
                    if (XPAY) {
                        float xv[24];
                        if constexpr (EARLY) {
#pragma unroll
                            for (int k = 0; k < 24; k++) xv[k] = xe[k];
                        } else {
                            load_spinor<PREC>((const char*)x_ + fb * (rhs0 + r), i, xv);
                        }
                        caxpy_f32<6>(cxur, cxui, xv, o);
                        caxpy_f32<6>(cxlr, cxli, xv + 12, o + 12);
                    }
                    if (EPI == EPI_RESID) {   // out_ is r: r -= alpha q, |r|^2 (q itself is never stored)
                        const float alpha = (float)cg->alpha[rhs0 + r];
                        float rv[24];
                        if constexpr (EARLY) {
#pragma unroll
                            for (int k = 0; k < 24; k++) rv[k] = rve[k];
                        } else {
                            load_spinor<PR, false>((const char*)out_ + fbo * (rhs0 + r), i, rv);   // coherent load: r is rewritten below
                        }
                        raxpy_f32<12>(-alpha, o, rv);
                        nrm[r] += norm2_site(rv);
                        store_spinor<PR>((char*)out_ + fbo * (rhs0 + r), i, rv);
                    } else {
                        store_spinor<PREC>((char*)out_ + fbo * (rhs0 + r), i, o);
                    }
                    if (EPI == EPI_NORM) {
                        if (PREC == TSM_BF16) {   // the norm of what was stored, i.e. of the vector the solver uses
                            float ob[24];
#pragma unroll
                            for (int k8 = 0; k8 < 3; k8++) { const uint4 pk = float_to_bf16x8(o + 8 * k8); bf16x8_to_float(pk, ob + 8 * k8); }
                            nrm[r] += norm2_site(ob);
                        } else {
                            nrm[r] += norm2_site(o);
                        }
                    }
                }
            }
            if (EPI != EPI_NONE && rhs0 < nrhs) {
                // sum over the row's 128 sites in a fixed order (A19): shuffle tree per warp, then the 4 warps;
                // only this row's 4 warps synchronise (named barrier), the other rows run on.  `red` is
                // double-buffered by group parity; a tile ends with __syncthreads().
                double* w = red + (ty * 2 + (grp & 1)) * 4 * R;
#pragma unroll
                for (int r = 0; r < R; r++) {
                    const double v = warp_sum(nrm[r]);
                    if ((tx & 31) == 0) w[(tx >> 5) * R + r] = v;
                }
                row_barrier(1 + ty, TT);
                if (tx < R) partials[(size_t)(rhs0 + tx) * ntiles + tile] = ((w[tx] + w[R + tx]) + w[2 * R + tx]) + w[3 * R + tx];
            }
        }
        __syncthreads();
    }
    if (EPI != EPI_NONE && fuse_reduce) {   // small lattices: the last block does k_cg_reduce's work (see dslash.cu)
        if (last_block_arrive(&cg->ticket)) {
            const int wid = (ty * TT + tx) >> 5;
            for (int j = wid; j < nrhs; j += 4 * RY) {
                const double v = sum_partials_warp(partials, j, ntiles);
                if ((tx & 31) == 0) cg_after_reduction(EPI == EPI_RESID ? 1 : 0, j, v, cg);
            }
        }
    }
}

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI, int RY, int R>
int launch_tile_t(tsm_ctx* ctx, int par, int nrhs, const void* pack, const void* in, const void* x, void* out, const DslashCoef& c,
                  int check_done)
{
    constexpr int NCH = RECON == 18 ? 36 : 24;
    const size_t SMEM = (size_t)2 * 4 * NCH * LB_ROW;   // two link buffers: the next tile's copy overlaps this tile's arithmetic (1 buffer: 799 vs 725 us)
    auto kern = k_dslash_tile<PREC, RECON, DAGGER, XPAY, EPI, RY, R>;
    static unsigned long long attr_done = 0;   // per device
    if (!((attr_done >> (ctx->device & 63)) & 1ull)) {
        TSM_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
        attr_done |= 1ull << (ctx->device & 63);
    }
    const Geom& g = ctx->g;
    const int ntiles = (g.Vh + TT - 1) / TT;
    const int slab = (g.S % TT == 0) ? 1 : 0;
    int grid = ctx->nsm;            // one CTA per SM (shared memory: two link buffers)
    if (grid > ntiles) grid = ntiles;
    if (EPI != EPI_NONE && (size_t)ntiles * nrhs > ctx->norm_partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const int pi = prof_begin(ctx, PREC, EPI == EPI_RESID ? 3 : (EPI == EPI_NORM ? 2 : (XPAY ? 1 : 0)), nrhs);
    const int fuse = (EPI != EPI_NONE && ntiles <= FUSE_NTILES) ? 1 : 0;
    kern<<<grid, dim3(TT, RY), SMEM, ctx->stream>>>(g, par, nrhs, ntiles, slab, pack, in, x, out, c, ctx->norm_partials, ctx->cg, check_done, fuse);
    prof_end(ctx, pi);
    ctx->launches++;
    ctx->norm_ntiles = ntiles;
    ctx->norm_reduced = fuse != 0;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

template <int PREC, int RECON, int RY, int R>
int launch_tile_v(tsm_ctx* ctx, int par, bool dagger, int nrhs, const void* pack, const void* in, const void* x, void* out,
                  const DslashCoef& c, int epi, int check_done)
{
    const bool xpay = x != nullptr;
#define GO(DG, XP, EP) return launch_tile_t<PREC, RECON, DG, XP, EP, RY, R>(ctx, par, nrhs, pack, in, x, out, c, check_done)
    if constexpr (!(RY == 3 && R == 1)) {   // plain launches: every shape but 3 x 1 (tile_shape)
        if (!dagger && !xpay && epi == EPI_NONE) GO(false, false, EPI_NONE);
        if (dagger && !xpay && epi == EPI_NONE) GO(true, false, EPI_NONE);
    }
    if constexpr (R == 1) {   // x term / epilogues: one source per thread
        if (!dagger && xpay && epi == EPI_NONE) GO(false, true, EPI_NONE);
        if (dagger && xpay && epi == EPI_NONE) GO(true, true, EPI_NONE);
        if (!dagger && xpay && epi == EPI_NORM) GO(false, true, EPI_NORM);
        if (dagger && xpay && epi == EPI_RESID) GO(true, true, EPI_RESID);
    }
#undef GO
    return tsm_fail(ctx, TSM_EINVAL, "unsupported dslash variant");
}

template <int PREC, int RECON>
int launch_tile_s(tsm_ctx* ctx, int ry, int r, int par, bool dagger, int nrhs, const void* pack, const void* in, const void* x,
                  void* out, const DslashCoef& c, int epi, int check_done)
{
#define SHAPE(RY_, R_) if (ry == RY_ && r == R_) return launch_tile_v<PREC, RECON, RY_, R_>(ctx, par, dagger, nrhs, pack, in, x, out, c, epi, check_done)
    SHAPE(4, 1);
    SHAPE(3, 2);
    SHAPE(2, 2);
    SHAPE(3, 1);
    SHAPE(2, 1);
    SHAPE(1, 1);
#undef SHAPE
    return tsm_fail(ctx, TSM_EINVAL, "unsupported tile shape");
}

}  // namespace

// Shape of the CTA for a batch of nrhs sources: RY source rows x R sources per thread; R divides nrhs.  A source's
// result is the same in every shape (the same operations in the same order per source).
static void tile_shape(int nrhs, bool plain, int& ry, int& r)
{
    if (nrhs == 1) { ry = 1; r = 1; return; }
    if (nrhs == 2) { ry = 2; r = 1; return; }
    if (plain && nrhs % 6 == 0) { ry = 3; r = 2; return; }
    if (plain && nrhs == 4) { ry = 2; r = 2; return; }   // config 4's batches: 65.7 us against 70.0 us for 4 x 1
    if (!plain && nrhs % 3 == 0) { ry = 3; r = 1; return; }
    ry = 4; r = 1;
}

// fp32 / bf16 storage, any nrhs >= 1.  mode bits as in launch_dslash.
int launch_dslash_tile(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x, void* out,
                       const DslashCoef& c, int mode)
{
    const int chk = (mode >> 1) & 1, nm = (mode & 4) ? EPI_RESID : ((mode & 1) ? EPI_NORM : EPI_NONE);
    int ry, r;
    tile_shape(nrhs, x == nullptr && nm == EPI_NONE, ry, r);
    const void* pack = ctx->gauge32[out_parity];
    if (prec == TSM_F32) {
        if (ctx->recon == 18) return launch_tile_s<TSM_F32, 18>(ctx, ry, r, out_parity, dagger, nrhs, pack, in, x, out, c, nm, chk);
        return launch_tile_s<TSM_F32, 12>(ctx, ry, r, out_parity, dagger, nrhs, pack, in, x, out, c, nm, chk);
    }
    if (prec == TSM_BF16) {
        if (ctx->recon == 18) return launch_tile_s<TSM_BF16, 18>(ctx, ry, r, out_parity, dagger, nrhs, pack, in, x, out, c, nm, chk);
        return launch_tile_s<TSM_BF16, 12>(ctx, ry, r, out_parity, dagger, nrhs, pack, in, x, out, c, nm, chk);
    }
    return tsm_fail(ctx, TSM_EINVAL, "tile stencil: unsupported precision");
}
