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
// One thread owns one output site of one source.  blockDim = (BS sites, RY sources): the warps
// of a block that differ only in the source index read the same link vectors, so links are
// fetched from HBM once per block and served from L1 for the other sources.
#include "reduce.cuh"

namespace {

template <typename T, int MU, int SGN> __device__ __forceinline__ void project(const T* p, T* h)
{
    // h = psi_up + SGN * a_mu psi_low, gamma_mu = [[0, a_mu], [a_mu^dag, 0]] (C3)
    constexpr T s = (T)SGN;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const T p0r = p[2 * c], p0i = p[2 * c + 1], p1r = p[6 + 2 * c], p1i = p[6 + 2 * c + 1];
        const T p2r = p[12 + 2 * c], p2i = p[12 + 2 * c + 1], p3r = p[18 + 2 * c], p3i = p[18 + 2 * c + 1];
        if (MU == 0) {          // a_0 = -i sigma_x
            h[2 * c] = p0r + s * p3i;      h[2 * c + 1] = p0i - s * p3r;
            h[6 + 2 * c] = p1r + s * p2i;  h[6 + 2 * c + 1] = p1i - s * p2r;
        } else if (MU == 1) {   // a_1 = -i sigma_y = [[0,-1],[1,0]]
            h[2 * c] = p0r - s * p3r;      h[2 * c + 1] = p0i - s * p3i;
            h[6 + 2 * c] = p1r + s * p2r;  h[6 + 2 * c + 1] = p1i + s * p2i;
        } else if (MU == 2) {   // a_2 = -i sigma_z = diag(-i, i)
            h[2 * c] = p0r + s * p2i;      h[2 * c + 1] = p0i - s * p2r;
            h[6 + 2 * c] = p1r - s * p3i;  h[6 + 2 * c + 1] = p1i + s * p3r;
        } else {                // a_3 = 1
            h[2 * c] = p0r + s * p2r;      h[2 * c + 1] = p0i + s * p2i;
            h[6 + 2 * c] = p1r + s * p3r;  h[6 + 2 * c + 1] = p1i + s * p3i;
        }
    }
}

template <typename T, int MU, int SGN> __device__ __forceinline__ void accumulate(const T* g, T* acc)
{
    // acc_up += g, acc_low += SGN * a_mu^dag g
    constexpr T s = (T)SGN;
#pragma unroll
    for (int k = 0; k < 12; k++) acc[k] += g[k];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const T g0r = g[2 * c], g0i = g[2 * c + 1], g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        if (MU == 0) {          // a_0^dag = i sigma_x
            acc[12 + 2 * c] -= s * g1i;  acc[12 + 2 * c + 1] += s * g1r;
            acc[18 + 2 * c] -= s * g0i;  acc[18 + 2 * c + 1] += s * g0r;
        } else if (MU == 1) {   // a_1^dag = [[0,1],[-1,0]]
            acc[12 + 2 * c] += s * g1r;  acc[12 + 2 * c + 1] += s * g1i;
            acc[18 + 2 * c] -= s * g0r;  acc[18 + 2 * c + 1] -= s * g0i;
        } else if (MU == 2) {   // a_2^dag = diag(i, -i)
            acc[12 + 2 * c] -= s * g0i;  acc[12 + 2 * c + 1] += s * g0r;
            acc[18 + 2 * c] += s * g1i;  acc[18 + 2 * c + 1] -= s * g1r;
        } else {
            acc[12 + 2 * c] += s * g0r;  acc[12 + 2 * c + 1] += s * g0i;
            acc[18 + 2 * c] += s * g1r;  acc[18 + 2 * c + 1] += s * g1i;
        }
    }
}

template <int PREC, int RECON, bool DAGGER, int MU>
__device__ __forceinline__ void hop_direction(const void* pack, const void* in, int Vh, int i, const int* nb,
                                              typename PT<PREC>::real ph_f, typename PT<PREC>::real ph_b,
                                              typename PT<PREC>::real* acc)
{
    using T = typename PT<PREC>::real;
    constexpr int SF = DAGGER ? +1 : -1;   // forward hop carries (1 - g_mu), dagger swaps
    T uf[18], ub[18], psi[24], h[12], gq[12];
    load_link_pair<PREC, RECON>(pack, Vh, i, MU, uf, ub);
    load_spinor<PREC>(in, Vh, nb[2 * MU], psi);
    project<T, MU, SF>(psi, h);
    if (MU == 3) {
#pragma unroll
        for (int k = 0; k < 12; k++) h[k] *= ph_f;
    }
    su3_mul(uf, h, gq);
    su3_mul(uf, h + 6, gq + 6);
    accumulate<T, MU, SF>(gq, acc);
    load_spinor<PREC>(in, Vh, nb[2 * MU + 1], psi);
    project<T, MU, -SF>(psi, h);
    if (MU == 3) {
#pragma unroll
        for (int k = 0; k < 12; k++) h[k] *= ph_b;
    }
    su3_mul(ub, h, gq);
    su3_mul(ub, h + 6, gq + 6);
    accumulate<T, MU, -SF>(gq, acc);
}

template <int PREC> struct DslashCfg {
    static constexpr int MAXT = (PREC == TSM_F64) ? 256 : 512;   // threads per block: 255 regs (fp64) / 128 regs (fp32)
};

// DOT: 0 none, 1: partial sums of Re<y, out>, last block leaves the totals in cg->pq[rhs].
template <int PREC, int RECON, bool DAGGER, bool XPAY, int DOT>
__global__ void __launch_bounds__(DslashCfg<PREC>::MAXT, 1)
k_dslash(const Geom g, const int par, const int nrhs, const void* __restrict__ pack, const void* __restrict__ in_,
         const void* __restrict__ x_, void* __restrict__ out_, const DslashCoef cf, const void* __restrict__ y_,
         double* __restrict__ partials, CgScalars* __restrict__ cg, const int check_done)
{
    using T = typename PT<PREC>::real;
    if (check_done && cg->all_done) return;
    const int rhs = blockIdx.y * blockDim.y + threadIdx.y;
    const int Vh = g.Vh;
    const size_t fb = field_bytes(PREC, Vh, 1);
    const char* in = (const char*)in_ + fb * rhs;
    const char* xin = XPAY ? (const char*)x_ + fb * rhs : nullptr;
    const char* yin = DOT ? (const char*)y_ + fb * rhs : nullptr;
    char* out = (char*)out_ + fb * rhs;
    const T cxur = (T)cf.x.up_re, cxui = (T)cf.x.up_im, cxlr = (T)cf.x.lo_re, cxli = (T)cf.x.lo_im;
    const T cdur = (T)cf.d.up_re, cdui = (T)cf.d.up_im, cdlr = (T)cf.d.lo_re, cdli = (T)cf.d.lo_im;
    double dot = 0.0;

    if (rhs < nrhs) {
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < Vh; i += gridDim.x * blockDim.x) {
            const SiteCoord s = decode_site(g, i, par);
            int nb[8];
            neighbours(g, i, s, nb);
            const T ph_f = (s.t == g.L[3] - 1) ? (T)g.theta : (T)1;
            const T ph_b = (s.t == 0) ? (T)g.theta : (T)1;
            T acc[24];
#pragma unroll
            for (int k = 0; k < 24; k++) acc[k] = 0;
            hop_direction<PREC, RECON, DAGGER, 0>(pack, in, Vh, i, nb, ph_f, ph_b, acc);
            hop_direction<PREC, RECON, DAGGER, 1>(pack, in, Vh, i, nb, ph_f, ph_b, acc);
            hop_direction<PREC, RECON, DAGGER, 2>(pack, in, Vh, i, nb, ph_f, ph_b, acc);
            hop_direction<PREC, RECON, DAGGER, 3>(pack, in, Vh, i, nb, ph_f, ph_b, acc);
            T o[24];
#pragma unroll
            for (int q = 0; q < 12; q++) {
                const T cr = (q < 6) ? cdur : cdlr, ci = (q < 6) ? cdui : cdli;
                o[2 * q] = cr * acc[2 * q] - ci * acc[2 * q + 1];
                o[2 * q + 1] = cr * acc[2 * q + 1] + ci * acc[2 * q];
            }
            if (XPAY) {
                T xv[24];
                load_spinor<PREC>(xin, Vh, i, xv);
#pragma unroll
                for (int q = 0; q < 12; q++) {
                    const T cr = (q < 6) ? cxur : cxlr, ci = (q < 6) ? cxui : cxli;
                    o[2 * q] += cr * xv[2 * q] - ci * xv[2 * q + 1];
                    o[2 * q + 1] += cr * xv[2 * q + 1] + ci * xv[2 * q];
                }
            }
            store_spinor<PREC>(out, Vh, i, o);
            if (DOT) {
                T yv[24];
                load_spinor<PREC>(yin, Vh, i, yv);
#pragma unroll
                for (int k = 0; k < 24; k++) dot += (double)yv[k] * (double)o[k];
            }
        }
    }
    if (DOT) {
        __shared__ double smem[32 * 8];
        const double tot = block_row_sum(dot, smem);
        if (threadIdx.x == 0 && rhs < nrhs) partials[(size_t)rhs * gridDim.x + blockIdx.x] = tot;
        if (last_block_arrive(&cg->ticket)) {
            const int flat = threadIdx.y * blockDim.x + threadIdx.x, nwarp = (blockDim.x * blockDim.y) >> 5;
            for (int r = flat >> 5; r < nrhs; r += nwarp) {
                const double v = sum_partials_warp(partials, r, gridDim.x);
                if ((flat & 31) == 0) cg->pq[r] = v;
            }
        }
    }
}

template <int PREC, int RECON, bool DAGGER, bool XPAY, int DOT>
int launch_t(tsm_ctx* ctx, int par, int nrhs, const void* pack, const void* in, const void* x, void* out,
             const DslashCoef& c, const void* y, int check_done)
{
    // 128 sites x RY sources per block.  The x extent and the x grid do not depend on the batch,
    // so every source sees the same thread->site map and the same reduction tree in any batch.
    const int bs = 128;
    const int max_ry = (PREC == TSM_F64) ? 2 : 4;     // register file: 512 x 128 regs (fp32), 256 x 255 (fp64)
    int ry = 1;
    if (nrhs % 4 == 0 && max_ry >= 4) ry = 4;          // RY sources share each link fetch through L1
    else if (nrhs % 2 == 0) ry = 2;
    dim3 block(bs, ry);
    const int gy = nrhs / ry;
    int gx = (ctx->g.Vh + bs - 1) / bs;
    const int cap = ctx->nsm * 8;                     // grid-stride beyond this; keeps the partial count small
    if (gx > cap) gx = cap;
    dim3 grid(gx, gy);
    if (DOT && (size_t)gx * nrhs > ctx->partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const int pi = prof_begin(ctx, PREC, DOT ? 2 : (XPAY ? 1 : 0), nrhs);
    k_dslash<PREC, RECON, DAGGER, XPAY, DOT><<<grid, block, 0, ctx->stream>>>(ctx->g, par, nrhs, pack, in, x, out, c, y,
                                                                             ctx->partials, ctx->cg, check_done);
    prof_end(ctx, pi);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

template <int PREC, int RECON>
int launch_p(tsm_ctx* ctx, int par, bool dagger, int nrhs, const void* pack, const void* in, const void* x, void* out,
             const DslashCoef& c, const void* y, int dot_mode, int check_done)
{
    const bool xpay = x != nullptr;
    const int dot = dot_mode != 0;
#define GO(DG, XP, DT) return launch_t<PREC, RECON, DG, XP, DT>(ctx, par, nrhs, pack, in, x, out, c, y, check_done)
    if (!dagger && !xpay && !dot) GO(false, false, 0);
    if (!dagger && xpay && !dot) GO(false, true, 0);
    if (dagger && !xpay && !dot) GO(true, false, 0);
    if (dagger && xpay && !dot) GO(true, true, 0);
    if (dagger && xpay && dot) GO(true, true, 1);
    if (!dagger && xpay && dot) GO(false, true, 1);
#undef GO
    return tsm_fail(ctx, TSM_EINVAL, "unsupported dslash variant");
}

}  // namespace

// dot_mode bit 0: Re<dot_y, out> into cg->pq; bit 1: early exit when cg->all_done.
int launch_dslash(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x,
                  void* out, const DslashCoef& c, const void* dot_y, int dot_mode)
{
    const int dm = dot_mode & 1, chk = (dot_mode >> 1) & 1;
    if (prec == TSM_F64)
        return launch_p<TSM_F64, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge64[out_parity], in, x, out, c, dot_y, dm, chk);
    if (prec == TSM_F32) {
        if (ctx->recon == 18)
            return launch_p<TSM_F32, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, dot_y, dm, chk);
        return launch_p<TSM_F32, 12>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, dot_y, dm, chk);
    }
    if (prec == TSM_BF16) {
        if (ctx->recon == 18)
            return launch_p<TSM_BF16, 18>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, dot_y, dm, chk);
        return launch_p<TSM_BF16, 12>(ctx, out_parity, dagger, nrhs, ctx->gauge32[out_parity], in, x, out, c, dot_y, dm, chk);
    }
    return tsm_fail(ctx, TSM_EINVAL, "bad precision");
}
