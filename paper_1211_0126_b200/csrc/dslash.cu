// dslash.cu -- H5: the even-odd twisted-mass Wilson hopping stencil with fused epilogues.
//
//   out(x) = Tx * xin(x) + Td * sum_mu [ phi+ U_mu(x) (1 -/+ g_mu) in(x+mu) + phi- U_mu(x-mu)^dag (1 +/- g_mu) in(x-mu) ]
//
// for x of one parity and `in` of the other (O2, O4 of DESIGN.md).  Upper sign:
// plain operator; lower sign (DAGGER): gamma5 D gamma5.  Tx, Td are "alpha + i beta gamma5" factors
// so that R^{+-1} and the kappa factors of Mhat ride along in the epilogue (the twisted term
// 1 + 2 i kappa mu gamma5 is never a separate pass).  Spin projection to 2 spin x 3 colour happens
// before the SU(3) multiply (C3); the time-boundary phase is applied in-kernel (A22).
//
// One thread owns one output site of one source.  blockDim = (128 sites, RY sources): the warps
// of a block that differ only in the source index read the same link vectors, so links are
// fetched once per block and served from L1 for the other sources.
#include <cstdlib>

#include "dslash_common.cuh"
#include "reduce.cuh"

namespace {

// NC: gather through the read-only path (ld.global.nc); false inside k_cg_persistent, where the gathered field is
// rewritten by other CTAs between two phases of the same launch
template <int PREC, int RECON, bool DAGGER, int MU, bool NC = true>
__device__ __forceinline__ void hop_direction(const void* pack, const void* in, int i, const int* nb,
                                              typename PT<PREC>::real ph_f, typename PT<PREC>::real ph_b,
                                              typename PT<PREC>::real* acc)
{
    using T = typename PT<PREC>::real;
    constexpr int SF = DAGGER ? +1 : -1;   // forward hop carries (1 - g_mu), dagger swaps
    T uf[18], ub[18], psi[24], h[12], gq[12];
    load_link_pair<PREC, RECON>(pack, i, MU, uf, ub);
    load_spinor<PREC, NC>(in, nb[2 * MU], psi);
    project<T, MU, SF>(psi, h);
    if (MU == 3 && ph_f != 1) {   // time-boundary phase (A22); skipping a multiplication by one is exact
        if constexpr (sizeof(T) == 4) rscale_f32<6>(ph_f, h);
        else {
#pragma unroll
            for (int k = 0; k < 12; k++) h[k] *= ph_f;
        }
    }
    su3_mul(uf, h, gq);
    su3_mul(uf, h + 6, gq + 6);
    accumulate<T, MU, SF>(gq, acc);
    load_spinor<PREC, NC>(in, nb[2 * MU + 1], psi);
    project<T, MU, -SF>(psi, h);
    if (MU == 3 && ph_b != 1) {
        if constexpr (sizeof(T) == 4) rscale_f32<6>(ph_b, h);
        else {
#pragma unroll
            for (int k = 0; k < 12; k++) h[k] *= ph_b;
        }
    }
    su3_mul(ub, h, gq);
    su3_mul(ub, h + 6, gq + 6);
    accumulate<T, MU, -SF>(gq, acc);
}

template <int PREC> struct DslashCfg {
    static constexpr int MAXT = (PREC == TSM_F64) ? 256 : 512;   // threads per block: 255 regs (fp64) / 128 regs (fp32)
};

constexpr int TILE = 128;   // sites per tile = blockDim.x

// Epilogue coefficients in the arithmetic type
template <typename T> struct SiteCoefs {
    T cxur, cxui, cxlr, cxli, cdur, cdui, cdlr, cdli;
    bool d_real;
};
template <typename T> __device__ __forceinline__ SiteCoefs<T> site_coefs(const DslashCoef& cf)
{
    SiteCoefs<T> c;
    c.cxur = (T)cf.x.up_re; c.cxui = (T)cf.x.up_im; c.cxlr = (T)cf.x.lo_re; c.cxli = (T)cf.x.lo_im;
    c.cdur = (T)cf.d.up_re; c.cdui = (T)cf.d.up_im; c.cdlr = (T)cf.d.lo_re; c.cdli = (T)cf.d.lo_im;
    c.d_real = c.cdui == 0 && c.cdli == 0;
    return c;
}

// The whole stencil for ONE output site (traversal index v) of ONE source: gather, hops, epilogue, store.  in / xf /
// out point at that source's fields.  Returns the site's contribution to the fused norm (EPI_NORM: |out|^2; EPI_RESID:
// |r|^2 after r -= alpha q).  Shared by k_dslash and the persistent CG kernel k_cg_persistent, so that the two give a
// source bit-identical results.
template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI, bool NC = true>
__device__ __forceinline__ double dslash_site(const Geom& g, const int par, const int slab, const int v, const void* pack, const char* in,
                                              const char* xf, char* out, const SiteCoefs<typename PT<PREC>::real>& c,
                                              const typename PT<PREC>::real alpha)
{
    using T = typename PT<PREC>::real;
    constexpr int PR = PREC == TSM_BF16 ? TSM_F32 : PREC;   // storage of r
    const T cxur = c.cxur, cxui = c.cxui, cxlr = c.cxlr, cxli = c.cxli, cdur = c.cdur, cdui = c.cdui, cdlr = c.cdlr, cdli = c.cdli;
    const bool d_real = c.d_real;
    double nrm = 0.0;
    {
        // slab order when whole tiles fit the z planes (S % 128 == 0), else plain cb order: in both
        // cases the same tiles, in the same order, as dslash_tile.cu (identical partial sums, A14/A19)
        SiteCoord s;
        int i = v;
        if (slab) i = traverse_site(g, v, par, s);
        else s = decode_site(g, v, par);
        int nb[8];
        neighbours(g, i, s, nb);
        const T ph_f = (s.t == g.L[3] - 1) ? (T)g.theta : (T)1;
        const T ph_b = (s.t == 0) ? (T)g.theta : (T)1;
        T acc[24];
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = 0;
        hop_direction<PREC, RECON, DAGGER, 0, NC>(pack, in, i, nb, ph_f, ph_b, acc);
        hop_direction<PREC, RECON, DAGGER, 1, NC>(pack, in, i, nb, ph_f, ph_b, acc);
        hop_direction<PREC, RECON, DAGGER, 2, NC>(pack, in, i, nb, ph_f, ph_b, acc);
        hop_direction<PREC, RECON, DAGGER, 3, NC>(pack, in, i, nb, ph_f, ph_b, acc);
        T o[24];
        if constexpr (sizeof(T) == 4) {   // packed fp32 (packed_f32.cuh): the same formulas
            if (d_real) { cscale_real_f32<6>(cdur, acc, o); cscale_real_f32<6>(cdlr, acc + 12, o + 12); }
            else { cscale_f32<6>(cdur, cdui, acc, o); cscale_f32<6>(cdlr, cdli, acc + 12, o + 12); }
            if (XPAY) {
                T xv[24];
                load_spinor<PREC, NC>(xf, i, xv);
                caxpy_f32<6>(cxur, cxui, xv, o);
                caxpy_f32<6>(cxlr, cxli, xv + 12, o + 12);
            }
        } else {
#pragma unroll
            for (int q = 0; q < 12; q++) {
                const T cr = (q < 6) ? cdur : cdlr, ci = (q < 6) ? cdui : cdli;
                if (d_real) {   // Td real (-kappa^2): the same values without the zero products
                    o[2 * q] = cr * acc[2 * q];
                    o[2 * q + 1] = cr * acc[2 * q + 1];
                } else {
                    o[2 * q] = cr * acc[2 * q] - ci * acc[2 * q + 1];
                    o[2 * q + 1] = cr * acc[2 * q + 1] + ci * acc[2 * q];
                }
            }
            if (XPAY) {
                T xv[24];
                load_spinor<PREC, NC>(xf, i, xv);
#pragma unroll
                for (int q = 0; q < 12; q++) {
                    const T cr = (q < 6) ? cxur : cxlr, ci = (q < 6) ? cxui : cxli;
                    o[2 * q] += cr * xv[2 * q] - ci * xv[2 * q + 1];
                    o[2 * q + 1] += cr * xv[2 * q + 1] + ci * xv[2 * q];
                }
            }
        }
        if (EPI == EPI_RESID) {
            T rv[24];
            load_spinor<PR, false>(out, i, rv);   // r is read and rewritten here: coherent load, not ld.global.nc
            if constexpr (sizeof(T) == 4) raxpy_f32<12>(-alpha, o, rv);
            else {
#pragma unroll
                for (int k = 0; k < 24; k++) rv[k] -= alpha * o[k];
            }
            nrm += norm2_site(rv);
            store_spinor<PR>(out, i, rv);
        } else {
            store_spinor<PREC>(out, i, o);
        }
        if (EPI == EPI_NORM) {
            if (PREC == TSM_BF16) {   // the norm of what was stored, i.e. of the vector the solver uses
                T ob[24];
#pragma unroll
                for (int k8 = 0; k8 < 3; k8++) { const uint4 pk = float_to_bf16x8((const float*)(o + 8 * k8)); bf16x8_to_float(pk, (float*)(ob + 8 * k8)); }
                nrm += norm2_site(ob);
            } else {
                nrm += norm2_site(o);
            }
        }
    }
    return nrm;
}

// Persistent kernel: gridDim.x resident blocks sweep the work items w = tile * gy + group in order,
// so the whole chip works on one narrow front of the traversal (tiles) and the gy source groups of a
// tile run next to each other in time (their link fetches meet in L2).  gridDim.x is a multiple of gy.
// EPI_NORM: the block also leaves sum |out|^2 of its tile, per source, in partials[rhs * ntiles + tile]
// (fixed tree, no atomics: the same value whatever the batch composition, A14/A19).
// EPI_RESID: the result q is not stored at all: `out` is the CG residual r (fp32 with bf16 storage), updated
// in place r -= alpha[rhs] * q, and the block leaves sum |r|^2 of its tile in partials (O5's "r -= alpha q;
// rr' = |r|^2" fused into the stencil that produces q).
template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI>
__global__ void __launch_bounds__(DslashCfg<PREC>::MAXT, 1)
k_dslash(const Geom g, const int par, const int gy, const int ntiles, const int slab, const void* __restrict__ pack,
         const void* __restrict__ in_, const void* __restrict__ x_, void* out_, const DslashCoef cf,
         double* __restrict__ partials, CgScalars* __restrict__ cg, const int check_done, const int fuse_reduce)
{
    using T = typename PT<PREC>::real;
    if (check_done && cg->all_done) return;
    const int Vh = g.Vh;
    constexpr int PR = PREC == TSM_BF16 ? TSM_F32 : PREC;   // storage of r
    const size_t fb = field_bytes(PREC, Vh, 1), fbo = field_bytes(EPI == EPI_RESID ? PR : PREC, Vh, 1);
    const SiteCoefs<T> sc = site_coefs<T>(cf);
    __shared__ double smem[EPI != EPI_NONE ? 32 * 4 : 1];

    for (int w = blockIdx.x; w < ntiles * gy; w += gridDim.x) {
        const int tile = w / gy, group = w - tile * gy;
        const int rhs = group * blockDim.y + threadIdx.y;
        const char* in = (const char*)in_ + fb * rhs;
        char* out = (char*)out_ + fbo * rhs;
        const int v = tile * TILE + threadIdx.x;
        double nrm = 0.0;
        if (v < Vh) {
            T alpha = 0;
            if (EPI == EPI_RESID) alpha = (T)cg->alpha[rhs];
            nrm = dslash_site<PREC, RECON, DAGGER, XPAY, EPI>(g, par, slab, v, pack, in, (const char*)x_ + fb * rhs, out, sc, alpha);
        }
        if (EPI != EPI_NONE) {
            const double tot = block_row_sum(nrm, smem);
            if (threadIdx.x == 0) partials[(size_t)rhs * ntiles + tile] = tot;
        }
    }
    // Lattices of at most FUSE_NTILES tiles: the last block of the grid to finish sums every source's partials (one
    // warp per source, an order that depends on ntiles only) and does what k_cg_reduce would -- there a separate
    // reduction launch costs half as much as the stencil itself.
    if (EPI != EPI_NONE && fuse_reduce) {
        if (last_block_arrive(&cg->ticket)) {
            const int wid = (threadIdx.y * blockDim.x + threadIdx.x) >> 5, nw = (blockDim.x * blockDim.y) >> 5;
            for (int j = wid; j < gy * (int)blockDim.y; j += nw) {
                const double v = sum_partials_warp(partials, j, ntiles);
                if ((threadIdx.x & 31) == 0) cg_after_reduction(EPI == EPI_RESID ? 1 : 0, j, v, cg);
            }
        }
    }
}

// resident blocks per SM of each instantiation, queried once
template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI> int resident_blocks(int threads)
{
    static int cache[5] = {0, 0, 0, 0, 0};   // indexed by blockDim.y
    const int ry = threads / TILE;
    if (cache[ry] == 0) {
        int nb = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_dslash<PREC, RECON, DAGGER, XPAY, EPI>, threads, 0) != cudaSuccess || nb < 1) nb = 1;
        cache[ry] = nb;
    }
    return cache[ry];
}

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI>
int launch_t(tsm_ctx* ctx, int par, int nrhs, const void* pack, const void* in, const void* x, void* out,
             const DslashCoef& c, int check_done)
{
    // 128 sites x RY sources per block: the RY warps rows read the same link vectors (L1 hits).
    const int max_ry = (PREC == TSM_F64) ? 2 : 4;     // register file: 512 x 128 regs (fp32), 256 x 255 (fp64)
    int ry = 1;
    if (nrhs % 4 == 0 && max_ry >= 4) ry = 4;
    else if (nrhs % 2 == 0) ry = 2;
    dim3 block(TILE, ry);
    const int gy = nrhs / ry;
    const int ntiles = (ctx->g.Vh + TILE - 1) / TILE;
    long long grid = (long long)ctx->nsm * resident_blocks<PREC, RECON, DAGGER, XPAY, EPI>(TILE * ry);
    grid -= grid % gy;
    if (grid < gy) grid = gy;
    if (grid > (long long)ntiles * gy) grid = (long long)ntiles * gy;
    if (EPI != EPI_NONE && (size_t)ntiles * nrhs > ctx->norm_partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const int pi = prof_begin(ctx, PREC, EPI == EPI_RESID ? 3 : (EPI == EPI_NORM ? 2 : (XPAY ? 1 : 0)), nrhs);
    const int fuse = (EPI != EPI_NONE && ntiles <= FUSE_NTILES) ? 1 : 0;
    k_dslash<PREC, RECON, DAGGER, XPAY, EPI><<<(unsigned)grid, block, 0, ctx->stream>>>(ctx->g, par, gy, ntiles, (ctx->g.S % TILE == 0) ? 1 : 0, pack, in, x, out, c,
                                                                                         ctx->norm_partials, ctx->cg, check_done, fuse);
    prof_end(ctx, pi);
    ctx->launches++;
    ctx->norm_ntiles = ntiles;
    ctx->norm_reduced = fuse != 0;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

template <int PREC, int RECON>
int launch_p(tsm_ctx* ctx, int par, bool dagger, int nrhs, const void* pack, const void* in, const void* x, void* out,
             const DslashCoef& c, int epi, int check_done)
{
    const bool xpay = x != nullptr;
#define GO(DG, XP, EP) return launch_t<PREC, RECON, DG, XP, EP>(ctx, par, nrhs, pack, in, x, out, c, check_done)
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

// Which kernel serves a stencil of precision prec in this context (1 k_dslash, 2 k_dslash_tile, 3 k_dslash_box,
// 5 k_dslash_small).  Automatic choice: on the smallest lattices (V_h <= SMALL_VH: configs 1, 2) every fp64 / fp32
// stencil, single sources and batches alike, goes to k_dslash_small (directions spread over warps: a latency, not a
// bandwidth, problem there); otherwise fp64 -> k_dslash; fp32 / bf16 -> k_dslash_tile for batches (nrhs >= 2) and
// k_dslash for single sources (those two give a source bit-identical results, A14).  k_dslash_box (fp32; 4-D tiles staged by tensor-map
// TMA) is correct on every lattice it accepts but measured slower than k_dslash_tile, so it
// runs only when asked for: tsm_set_stencil_kernel(ctx, 3) sends EVERY fp32 stencil of the context to it, single
// sources included, so that a source's result still does not depend on its batch.
constexpr int SMALL_VH = 16384;   // measured: +19 % LP solves/s at 4^3 x 8, +9 % at 8^3 x 16, -15 % at 16^3 x 32 (V_h = 65 536)
static int stencil_kernel_for(const tsm_ctx* ctx, int prec, int nrhs)
{
    if (ctx->stencil_choice == 0 && prec != TSM_BF16 && ctx->g.Vh <= SMALL_VH) return 5;
    if (ctx->stencil_choice == 5 && prec != TSM_BF16) return 5;
    if (prec == TSM_F64) return 1;
    const bool box_ok = prec == TSM_F32 && box_stencil_supported(ctx);
    if (ctx->stencil_choice == 1) return 1;
    if (ctx->stencil_choice == 2) return 2;
    if (ctx->stencil_choice == 3 && box_ok) return 3;
    return nrhs >= 2 ? 2 : 1;
}

// mode bit 0: leave per-tile sums of |out|^2 in ctx->partials (the CG's <p, Mhat^dag Mhat p> = |Mhat p|^2);
// bit 1: early exit when cg->all_done; bit 2: `out` is the CG residual, updated in place (EPI_RESID).
int launch_dslash(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x,
                  void* out, const DslashCoef& c, int mode)
{
    const int chk = (mode >> 1) & 1, nm = (mode & 4) ? EPI_RESID : ((mode & 1) ? EPI_NORM : EPI_NONE);
    const int which = stencil_kernel_for(ctx, prec, nrhs);
    if (which == 5) return launch_dslash_small(ctx, prec, out_parity, dagger, nrhs, in, x, out, c, mode);
    if (which == 3) return launch_dslash_box(ctx, out_parity, dagger, nrhs, in, x, out, c, mode);
    if (which == 2) return launch_dslash_tile(ctx, prec, out_parity, dagger, nrhs, in, x, out, c, mode);
    if (prec == TSM_F64)
        return launch_p<TSM_F64, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge64[out_parity], in, x, out, c, nm, chk);
    if (prec == TSM_F32) {
        if (ctx->recon == 18)
            return launch_p<TSM_F32, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, nm, chk);
        return launch_p<TSM_F32, 12>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, nm, chk);
    }
    if (prec == TSM_BF16) {
        if (ctx->recon == 18)
            return launch_p<TSM_BF16, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, nm, chk);
        return launch_p<TSM_BF16, 12>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, nm, chk);
    }
    return tsm_fail(ctx, TSM_EINVAL, "bad precision");
}

extern "C" const char* tsm_stencil_kernel_name(const tsm_ctx* ctx, int prec, int nrhs)
{
    if (!ctx || prec < 0 || prec > TSM_BF16 || nrhs < 1) return "none";
    const int which = stencil_kernel_for(ctx, prec, nrhs);
    return which == 5 ? "k_dslash_small" : (which == 3 ? "k_dslash_box" : (which == 2 ? "k_dslash_tile" : "k_dslash"));
}

extern "C" int tsm_set_stencil_kernel(tsm_ctx* ctx, int which)
{
    if (!ctx) return TSM_EINVAL;
    if (which < 0 || which > 5 || which == 4)
        return tsm_fail(ctx, TSM_EINVAL, "stencil kernel: 0 automatic, 1 k_dslash, 2 k_dslash_tile, 3 k_dslash_box, 5 k_dslash_small");
    if (which != ctx->stencil_choice) ctx_drop_graphs(ctx);   // captured CG iterations hold the old kernels
    ctx->stencil_choice = which;
    return TSM_OK;
}

// ------------------------------------------------------------------ launch-free CG for lattices that fit in L2
// (hard part 4).  On 4^3 x 8 .. 16^3 x 32 a CG iteration is five kernels of
// 6-12 us each whose time is launch latency and dependent-load chains, not bandwidth.  k_cg_persistent runs the WHOLE
// iteration loop of O5 in one cooperative launch: a co-resident grid of 128-thread CTAs sweeps the 128-site tiles, the
// four stencil phases and the x / p update are separated by grid-wide barriers (cooperative groups), the two dot
// products are summed redundantly by every CTA from the per-tile partials (no atomics), and the stopping test is
// evaluated on the device.  Every phase is the same code as the kernel-by-kernel path: dslash_site() for the stencils,
// block_row_sum() per tile, sum_partials_warp()'s order over tiles, k_cg_update_xp's update formula -- so a source's
// iterate is bit-identical to the one k_dslash / k_dslash_tile + k_cg_update_xp produce (lattices of at most
// FUSE_NTILES tiles, where those kernels sum their tiles in this same order).
#include <cooperative_groups.h>

namespace {

namespace cgp = cooperative_groups;

template <int PREC, int RECON, bool DAGGER, bool XPAY, int EPI>
__device__ __forceinline__ void pcg_stencil(const PcgArgs& a, const int par, const void* in_, const void* x_, void* out_, const DslashCoef& cf,
                                            const double* s_alpha, double* partials, double* smem)
{
    using T = typename PT<PREC>::real;
    const int Vh = a.g.Vh;
    const size_t fb = field_bytes(PREC, Vh, 1);
    const SiteCoefs<T> sc = site_coefs<T>(cf);
    for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const int v = tile * TILE + threadIdx.x;
        for (int rhs = 0; rhs < a.nrhs; rhs++) {
            double nrm = 0.0;
            if (v < Vh) {
                T alpha = 0;
                if (EPI == EPI_RESID) alpha = (T)s_alpha[rhs];
                nrm = dslash_site<PREC, RECON, DAGGER, XPAY, EPI, false>(a.g, par, a.slab, v, a.pack[par], (const char*)in_ + fb * rhs,
                                                                  (const char*)x_ + fb * rhs, (char*)out_ + fb * rhs, sc, alpha);
            }
            if (EPI != EPI_NONE) {
                const double tot = block_row_sum(nrm, smem);   // blockDim.y == 1: the tree of k_dslash's source row
                if (threadIdx.x == 0) partials[(size_t)rhs * a.ntiles + tile] = tot;
            }
        }
    }
}

template <int PREC, int RECON>
__global__ void __launch_bounds__(TILE, PREC == TSM_F64 ? 2 : 4) k_cg_persistent(const PcgArgs a)
{
    using T = typename PT<PREC>::real;
    cgp::grid_group grid = cgp::this_grid();
    __shared__ double smem[32];
    __shared__ double s_alpha[TSM_MAX_NRHS], s_rr[TSM_MAX_NRHS], s_rrnew[TSM_MAX_NRHS], s_beta[TSM_MAX_NRHS], s_pq[TSM_MAX_NRHS];
    __shared__ int s_done[TSM_MAX_NRHS], s_iters[TSM_MAX_NRHS], s_status[TSM_MAX_NRHS];
    __shared__ int s_all, s_broke;
    CgScalars* cg = a.cg;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int Vh = a.g.Vh, nrhs = a.nrhs;
    // every CTA keeps its own copy of the per-source scalars: all CTAs derive the same values from the same partials
    if (tid < nrhs) {
        s_rr[tid] = cg->rr[tid]; s_done[tid] = cg->done[tid]; s_iters[tid] = cg->iters[tid]; s_status[tid] = cg->status[tid];
        s_beta[tid] = cg->beta[tid]; s_pq[tid] = cg->pq[tid]; s_alpha[tid] = 0.0; s_rrnew[tid] = cg->rr_new[tid];
    }
    if (tid == 0) { s_all = cg->all_done; s_broke = 0; }
    __syncthreads();
    double* part_w = a.partials;
    double* part_r = a.partials + (size_t)nrhs * a.ntiles;

    for (int it = 0; it < a.max_iter && !s_all; it++) {
        pcg_stencil<PREC, RECON, false, false, EPI_NONE>(a, 1, a.p, nullptr, a.t, a.c1, s_alpha, nullptr, smem);   // t = R^-1 D_oe p
        grid.sync();
        pcg_stencil<PREC, RECON, false, true, EPI_NORM>(a, 0, a.t, a.p, a.w, a.c2, s_alpha, part_w, smem);         // w = Mhat p; |w|^2 per tile
        grid.sync();
        for (int j = wid; j < nrhs; j += TILE / 32) {   // alpha = rr / |w|^2 (cg_after_reduction, which == 0)
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
        pcg_stencil<PREC, RECON, true, false, EPI_NONE>(a, 1, a.w, nullptr, a.t, a.c3, s_alpha, nullptr, smem);    // t = Rb^-1 D_oe^dag w
        grid.sync();
        pcg_stencil<PREC, RECON, true, true, EPI_RESID>(a, 0, a.t, a.w, a.r, a.c4, s_alpha, part_r, smem);         // r -= alpha Mhat^dag w; |r|^2 per tile
        grid.sync();
        for (int j = wid; j < nrhs; j += TILE / 32) {   // rr' (which == 1)
            const double v = sum_partials_warp(part_r, j, a.ntiles);
            if (lane == 0) s_rrnew[j] = v;
        }
        __syncthreads();
        // x += alpha p; p = r + beta p on this CTA's own tiles (k_cg_update_xp's formula; element-wise, any site order)
        const size_t fb = field_bytes(PREC, Vh, 1);
        for (int rhs = 0; rhs < nrhs; rhs++) {
            if (s_done[rhs]) continue;
            const T alpha = (T)s_alpha[rhs];
            const T beta = (T)(s_rrnew[rhs] / s_rr[rhs]);
            char* x = (char*)a.x + fb * rhs;
            char* p = (char*)a.p + fb * rhs;
            const char* r = (const char*)a.r + fb * rhs;
            for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
                const int i = tile * TILE + tid;   // cb index: the update does not care about the traversal order
                if (i >= Vh) continue;
#pragma unroll
                for (int k8 = 0; k8 < 3; k8++) {
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
                    if (a.tol > 0 && sqrt(v / cg->bb[j]) <= a.tol) s_done[j] = 1;
                }
                all &= s_done[j];
            }
            s_all = all;
        }
        grid.sync();   // p is complete (and s_all visible to this CTA's threads) before the next iteration gathers it
    }
    if (blockIdx.x == 0) {
        __syncthreads();
        if (tid < nrhs) {
            cg->rr[tid] = s_rr[tid]; cg->done[tid] = s_done[tid]; cg->iters[tid] = s_iters[tid]; cg->status[tid] = s_status[tid];
            cg->beta[tid] = s_beta[tid]; cg->pq[tid] = s_pq[tid]; cg->alpha[tid] = s_alpha[tid]; cg->rr_new[tid] = s_rrnew[tid];
        }
        if (tid == 0) {
            cg->all_done = s_all;
            if (s_broke) cg->sticky_breakdown = 1;
        }
    }
}

template <int PREC, int RECON> int launch_pcg_t(tsm_ctx* ctx, PcgArgs& a)
{
    auto kern = k_cg_persistent<PREC, RECON>;
    static int resident[64] = {0};   // co-resident CTAs per SM of this instantiation, per device
    if (ctx->device >= 64) return tsm_fail(ctx, TSM_EINVAL, "persistent CG: device index beyond 63");
    if (!resident[ctx->device]) {
        int nb = 0;
        TSM_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, TILE, 0));
        if (nb < 1) return tsm_fail(ctx, TSM_ECUDA, "persistent CG kernel does not fit an SM");
        resident[ctx->device] = nb;
    }
    int grid = ctx->nsm * resident[ctx->device];
    if (grid > a.ntiles) grid = a.ntiles;
    void* params[] = {(void*)&a};
    TSM_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(TILE), params, 0, ctx->stream));
    ctx->launches++;
    return TSM_OK;
}

}  // namespace

// Lattices the persistent solver serves: at most FUSE_NTILES tiles (the kernel-by-kernel path then sums its tiles in the
// same order) and room in the reduction scratch for two sets of partials.
bool cg_persistent_supported(const tsm_ctx* ctx, int prec, int nrhs)
{
    const int ntiles = (ctx->g.Vh + TILE - 1) / TILE;
    return (prec == TSM_F64 || prec == TSM_F32) && ntiles <= FUSE_NTILES && (size_t)2 * nrhs * ntiles <= ctx->norm_partials_count;
}

// Where the persistent solver is the better choice (measured): the lattices whose stencil is
// k_dslash_small (+34 % / +42 % LP solves/s at 4^3 x 8 / 8^3 x 16); with 128-site tiles it loses (-12 % at 16^3 x 32).
bool cg_persistent_preferred(const tsm_ctx* ctx, int prec, int nrhs)
{
    return cg_persistent_supported(ctx, prec, nrhs) && stencil_kernel_for(ctx, prec, nrhs) == 5;
}

// max_iter iterations of O5 (or until every source is frozen) in ONE cooperative launch.  c1..c4: the coefficient pairs of
// the four stencil launches of cg_iteration, in order.
int launch_cg_persistent(tsm_ctx* ctx, int prec, int nrhs, void* x, void* r, void* p, void* w, void* t, const DslashCoef& c1,
                         const DslashCoef& c2, const DslashCoef& c3, const DslashCoef& c4, double tol, int max_iter, const PcgArgs* whole)
{
    if (!cg_persistent_supported(ctx, prec, nrhs)) return tsm_fail(ctx, TSM_EINVAL, "persistent CG: lattice or precision not supported");
    PcgArgs a;
    a.g = ctx->g;
    a.nrhs = nrhs;
    const bool small = stencil_kernel_for(ctx, prec, nrhs) == 5;   // where k_dslash_small is the stencil, its persistent form
    a.ntiles = small ? (int)(padded_sites(ctx->g.Vh) / LB) : (ctx->g.Vh + TILE - 1) / TILE;
    a.slab = (ctx->g.S % TILE == 0) ? 1 : 0;
    a.max_iter = max_iter;
    a.tol = tol;
    a.x = x; a.r = r; a.p = p; a.w = w; a.t = t;
    a.c1 = c1; a.c2 = c2; a.c3 = c3; a.c4 = c4;
    a.partials = ctx->norm_partials;
    a.cg = ctx->cg;
    a.whole = 0;
    a.s_o = a.aux = nullptr;
    a.init_groups = nullptr;
    a.init_gx = 0;
    if (whole) {   // source preparation, CG initialisation and reconstruction in the same launch (small form only)
        a.whole = 1;
        a.s_o = whole->s_o; a.aux = whole->aux; a.tw_rinv = whole->tw_rinv;
        a.cp1 = whole->cp1; a.cp2 = whole->cp2; a.cp3 = whole->cp3; a.crec = whole->crec;
        a.init_groups = ctx->partials;
        a.init_gx = blas_grid_x(ctx);
        // k_cg_init's summation order can be reproduced only where each of its threads holds at most one item
        if (!small || (size_t)nrhs * 3 * a.ntiles > ctx->partials_count || (long long)a.init_gx * 256 < 3LL * padded_sites(ctx->g.Vh))
            return tsm_fail(ctx, TSM_EINVAL, "persistent CG: the whole-solve form does not apply to this lattice");
    }
    ctx->norm_reduced = false;
    if (prec == TSM_F64) {
        a.pack[0] = ctx->gauge64[0]; a.pack[1] = ctx->gauge64[1];
    } else {
        a.pack[0] = ctx->gauge32[0]; a.pack[1] = ctx->gauge32[1];
    }
    if (small) return launch_cg_persistent_small(ctx, prec, a);
    if (prec == TSM_F64) return launch_pcg_t<TSM_F64, 18>(ctx, a);
    if (ctx->recon == 18) return launch_pcg_t<TSM_F32, 18>(ctx, a);
    return launch_pcg_t<TSM_F32, 12>(ctx, a);
}
