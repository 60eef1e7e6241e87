// contract.cu -- H8-H10: per-timeslice loop contractions and the TSM accumulators.
//
// H8  C_{ab}(t) = sum_{x in t, c} conj(eta_{ac}(x)) s_{bc}(x); L_Gamma(t) = sum_{ab} Gamma_{ab} C_{ab}(t)
//     ("(1/N) sum <eta^dag X s>", "all possible insertion times"; O6).
// H9  the same with s replaced by (D_mu s)(x) = 1/2 [phi+ U_mu(x) s(x+mu) - phi- U_mu(x-mu)^dag s(x-mu)]
//     for mu = 0..3 (reading A18; O6b).
// eta is never read from memory: it is regenerated from the Philox counter (PAPER.md:80,
// "noise sources were generated on-the-fly").  Sums are fp64 with a fixed tree (A19).
// N1  one-end trick (Eq. 2.5; reading A24): the same 4x4 spin matrix with eta replaced by s
//     itself, C'_{ab}(t) = sum_{x in t, c} conj(s_{ac}(x)) s_{bc}(x), then
//     L1_Gamma(t) = -2 i a sum_{ab} (gamma5 Gamma)_{ab} C'_{ab}(t), a = 2 kappa mu, whose noise average is
//     sum_{x in t} tr[Gamma (M_u^-1 - M_d^-1)(x,x)].
// N2  generalised one-end trick (Eq. 2.6): y = D_W s with D_W = M(mu = 0) = 1 - kappa D_hop
//     (two stencil launches into a scratch field), C''_{ab}(t) = sum conj(s_{ac}) y_{bc},
//     L2_Gamma(t) = 2 sum_{ab} (gamma5 Gamma gamma5)_{ab} C''_{ab}(t); noise average
//     sum_{x in t} tr[Gamma (M_u^-1 + M_d^-1)(x,x)].
// N3  momentum-projected local loops (PAPER.md:72 uses cuFFT for the Fourier transform; reading A25): for a
//     short list of integer momenta n, L_Gamma(t, p) = sum_{x in t} exp(+2 pi i n.x/L) eta^dag Gamma s, as one
//     more block group per momentum (a direct phase sum: a handful of momenta, not a full FFT).
// H10 Eq. 2.4 accumulators (O7).
#include "reduce.cuh"

namespace {

constexpr int CT_BS = 128;
constexpr int CT_MAXBLK = 8;   // blocks per (timeslice, parity)

// grid = (nblk * ngroup_in_launch, Lt, nrhs * 2); MODE 0: local; 1: derivative, mu = blockIdx.x / nblk; 2: one-end;
// 3: generalised one-end (second = D_W s, same [parity][rhs] layout as sol).
// 4: momentum-projected local, momentum index = blockIdx.x / nblk.
// partials: [rhs][group][t][par][blk][32], group 0 local, 1..4 derivative mu, 5 one-end, 6 generalised one-end,
// 7 + m momentum m
constexpr int CT_NGROUP = 7 + TSM_MAX_MOMENTA;
enum { CT_LOCAL = 0, CT_DERIV = 1, CT_ONE_END = 2, CT_GEN_ONE_END = 3, CT_MOMENTUM = 4 };
struct Momenta { int n[TSM_MAX_MOMENTA][3]; };
template <int PREC, int RECON, int MODE>
__global__ void __launch_bounds__(CT_BS) k_contract(const Geom g, const int nrhs, const int nblk, const void* __restrict__ sol,
                                                    const void* __restrict__ second, const void* __restrict__ pack0, const void* __restrict__ pack1,
                                                    const uint64_t seed, const uint32_t* __restrict__ ids, const int kind,
                                                    double* __restrict__ partials, const Momenta mom)
{
    using T = typename PT<PREC>::real;
    const int Vh = g.Vh;
    const int blk = blockIdx.x % nblk, mu = blockIdx.x / nblk;
    const int t = blockIdx.y;
    const int rhs = blockIdx.z >> 1, par = blockIdx.z & 1;
    const size_t fpar = field_bytes(PREC, Vh, nrhs), frhs = field_bytes(PREC, Vh, 1);
    const char* s_same = (const char*)sol + fpar * par + frhs * rhs;
    const char* s_other = (const char*)sol + fpar * (1 - par) + frhs * rhs;
    const void* pack = par ? pack1 : pack0;
    const uint32_t sid = ids[rhs];

    double C[32];
#pragma unroll
    for (int k = 0; k < 32; k++) C[k] = 0;

    for (int j = blk * CT_BS + threadIdx.x; j < g.Vsh; j += nblk * CT_BS) {
        const int i = t * g.Vsh + j;
        const SiteCoord sc = decode_site(g, i, par);
        uint32_t bits = 0;
        if (MODE == CT_LOCAL || MODE == CT_DERIV || MODE == CT_MOMENTUM) bits = noise_bits(lex_of_site(g, sc), seed, sid, kind);
        T v[24], sv[24];
        if (MODE == CT_GEN_ONE_END) {
            load_spinor<PREC>(s_same, i, sv);
            load_spinor<PREC>((const char*)second + fpar * par + frhs * rhs, i, v);
        } else if (MODE != CT_DERIV) {
            load_spinor<PREC>(s_same, i, v);
        } else {
            int nb[8];
            neighbours(g, i, sc, nb);
            T uf[18], ub[18], sf[24], sb[24], a[6], b[6];
            // runtime mu: the four directions are four block groups of the same launch
            switch (mu) {
                case 0: load_link_pair<PREC, RECON>(pack, i, 0, uf, ub); break;
                case 1: load_link_pair<PREC, RECON>(pack, i, 1, uf, ub); break;
                case 2: load_link_pair<PREC, RECON>(pack, i, 2, uf, ub); break;
                default: load_link_pair<PREC, RECON>(pack, i, 3, uf, ub); break;
            }
            load_spinor<PREC>(s_other, nb[2 * mu], sf);
            load_spinor<PREC>(s_other, nb[2 * mu + 1], sb);
            const T ph_f = (mu == 3 && sc.t == g.L[3] - 1) ? (T)g.theta : (T)1;
            const T ph_b = (mu == 3 && sc.t == 0) ? (T)g.theta : (T)1;
#pragma unroll
            for (int al = 0; al < 4; al++) {
                su3_mul(uf, sf + 6 * al, a);
                su3_mul(ub, sb + 6 * al, b);
#pragma unroll
                for (int k = 0; k < 6; k++) v[6 * al + k] = (T)0.5 * (ph_f * a[k] - ph_b * b[k]);
            }
        }
        if (MODE == CT_MOMENTUM) {   // s <- exp(2 pi i n.x/L) s; the fraction is reduced in integers first
            const int x = 2 * sc.xh + sc.rowpar;
            const double fr = (double)(((long long)mom.n[mu][0] * x) % g.L[0]) / g.L[0] +
                              (double)(((long long)mom.n[mu][1] * sc.y) % g.L[1]) / g.L[1] +
                              (double)(((long long)mom.n[mu][2] * sc.z) % g.L[2]) / g.L[2];
            double sn, cs;
            sincospi(2.0 * fr, &sn, &cs);
#pragma unroll
            for (int q = 0; q < 12; q++) {
                const double re = (double)v[2 * q], im = (double)v[2 * q + 1];
                v[2 * q] = (T)(cs * re - sn * im);
                v[2 * q + 1] = (T)(cs * im + sn * re);
            }
        }
#pragma unroll
        for (int al = 0; al < 4; al++)
#pragma unroll
            for (int c = 0; c < 3; c++) {
                double cr, ci;
                if (MODE == CT_ONE_END) {   // conj(s) in place of conj(eta)
                    cr = (double)v[2 * (3 * al + c)];
                    ci = -(double)v[2 * (3 * al + c) + 1];
                } else if (MODE == CT_GEN_ONE_END) {
                    cr = (double)sv[2 * (3 * al + c)];
                    ci = -(double)sv[2 * (3 * al + c) + 1];
                } else {
                    float er, ei;
                    noise_value((bits >> (2 * (3 * al + c))) & 3, kind, er, ei);
                    cr = er;
                    ci = -ei;   // conj(eta)
                }
#pragma unroll
                for (int be = 0; be < 4; be++) {
                    const double sr = (double)v[2 * (3 * be + c)], si = (double)v[2 * (3 * be + c) + 1];
                    C[2 * (4 * al + be)] += cr * sr - ci * si;
                    C[2 * (4 * al + be) + 1] += cr * si + ci * sr;
                }
            }
    }
    // block reduction of the 32 sums: shuffle tree per warp, fixed serial sum over warps
    __shared__ double sm[CT_BS / 32][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 32; k++) {
        const double r = warp_sum(C[k]);
        if (lane == 0) sm[w][k] = r;
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        double tot = 0;
        for (int ww = 0; ww < CT_BS / 32; ww++) tot += sm[ww][threadIdx.x];
        const int group = MODE == CT_DERIV ? 1 + mu : (MODE == CT_ONE_END ? 5 : (MODE == CT_GEN_ONE_END ? 6 : (MODE == CT_MOMENTUM ? 7 + mu : 0)));
        const size_t o = ((((size_t)rhs * CT_NGROUP + group) * g.L[3] + t) * 2 + par) * nblk + blk;
        partials[o * 32 + threadIdx.x] = tot;
    }
}

// grid = (Lt, 6, nrhs), 32 threads: finish the sums and apply the 16 Gamma.  op_base[group] is the first op
// index of the group, or -1 if the group is not computed; two_a = 2 * (2 kappa mu) for the one-end group.
struct OpBase { int v[CT_NGROUP]; };
__global__ void k_contract_finish(const int Lt, const int nblk, const int n_ops, const GammaTable gt, const OpBase ob,
                                  const double two_a, const double* __restrict__ partials, double* __restrict__ loops)
{
    const int t = blockIdx.x, group = blockIdx.y, rhs = blockIdx.z, k = threadIdx.x;
    if (ob.v[group] < 0) return;
    __shared__ double C[32];
    double tot = 0;
    for (int pb = 0; pb < 2 * nblk; pb++) {
        const size_t o = (((size_t)rhs * CT_NGROUP + group) * Lt + t) * 2 * nblk + pb;
        tot += partials[o * 32 + k];
    }
    C[k] = tot;
    __syncthreads();
    if (k < 16) {
        double re = 0, im = 0;
        for (int al = 0; al < 4; al++) {
            const int be = gt.col[k][al];
            // one-end: (gamma5 Gamma)_{al,be} = +-Gamma_{al,be} (gamma5 = diag(1,1,-1,-1): phase + 2 on rows 2,3)
            // generalised one-end: (gamma5 Gamma gamma5)_{al,be}: one more sign when be is a lower spin
            const int ph = (gt.ph[k][al] + (((group == 5 || group == 6) && al >= 2) ? 2 : 0) + ((group == 6 && be >= 2) ? 2 : 0)) & 3;
            const double cr = C[2 * (4 * al + be)], ci = C[2 * (4 * al + be) + 1];
            // multiply by i^ph
            re += (ph == 0) ? cr : (ph == 1) ? -ci : (ph == 2) ? -cr : ci;
            im += (ph == 0) ? ci : (ph == 1) ? cr : (ph == 2) ? -ci : -cr;
        }
        double* dst = loops + (((size_t)rhs * n_ops + ob.v[group] + k) * Lt + t) * 2;
        if (group == 5) {   // times -2 i a:  -2ia (re + i im) = 2a im - i 2a re
            dst[0] = two_a * im;
            dst[1] = -two_a * re;
        } else if (group == 6) {   // times 2 (Eq. 2.6)
            dst[0] = 2.0 * re;
            dst[1] = 2.0 * im;
        } else {
            dst[0] = re;
            dst[1] = im;
        }
    }
}

// acc += a[r] - b[r] source by source, in source order: the sums of Eq. 2.4 come out bit-identical
// however the sources were batched (b == nullptr: acc += a[r]).
__global__ void k_accumulate(const int n, const int nrhs, double* __restrict__ acc, const double* __restrict__ a, const double* __restrict__ b)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    double s = acc[idx];
    for (int r = 0; r < nrhs; r++) s += b ? (a[(size_t)r * n + idx] - b[(size_t)r * n + idx]) : a[(size_t)r * n + idx];
    acc[idx] = s;
}

__global__ void k_finalize(const int n, const double* __restrict__ corr, const double* __restrict__ lp, const double w_hp,
                           const double w_lp, double* __restrict__ out)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < n) out[idx] = w_hp * corr[idx] + w_lp * lp[idx];
}

}  // namespace

// The CUDA path's own Gamma tables: each Gamma is a monomial matrix, Gamma_{a, col[a]} = i^ph[a].
// gamma_mu are typed from C3 (gamma_k = [[0,-i sigma_k],[i sigma_k,0]], gamma_3 = [[0,1],[1,0]]);
// gamma5 gamma_mu and sigma_{mu nu} = i gamma_mu gamma_nu (mu != nu) follow by monomial products.
void build_gamma_table(GammaTable& t)
{
    struct Mono { int col[4]; int ph[4]; };
    auto mul = [](const Mono& a, const Mono& b) {   // (AB)_{r, b.col[a.col[r]]} = a.ph[r] * b.ph[a.col[r]]
        Mono o;
        for (int r = 0; r < 4; r++) { o.col[r] = b.col[a.col[r]]; o.ph[r] = (a.ph[r] + b.ph[a.col[r]]) & 3; }
        return o;
    };
    const Mono one = {{0, 1, 2, 3}, {0, 0, 0, 0}};
    const Mono g5 = {{0, 1, 2, 3}, {0, 0, 2, 2}};
    const Mono gm[4] = {
        {{3, 2, 1, 0}, {3, 3, 1, 1}},   // gamma_0: rows (0:-i@3, 1:-i@2, 2:+i@1, 3:+i@0)
        {{3, 2, 1, 0}, {2, 0, 0, 2}},   // gamma_1: (-1@3, +1@2, +1@1, -1@0)
        {{2, 3, 0, 1}, {3, 1, 1, 3}},   // gamma_2: (-i@2, +i@3, +i@0, -i@1)
        {{2, 3, 0, 1}, {0, 0, 0, 0}},   // gamma_3
    };
    const Mono eye_i = {{0, 1, 2, 3}, {1, 1, 1, 1}};   // i * 1
    Mono all[16];
    all[0] = one;
    all[1] = g5;
    for (int m = 0; m < 4; m++) { all[2 + m] = gm[m]; all[6 + m] = mul(g5, gm[m]); }
    const int pr[6][2] = {{0, 1}, {0, 2}, {0, 3}, {1, 2}, {1, 3}, {2, 3}};
    for (int k = 0; k < 6; k++) all[10 + k] = mul(eye_i, mul(gm[pr[k][0]], gm[pr[k][1]]));
    for (int G = 0; G < 16; G++)
        for (int r = 0; r < 4; r++) { t.col[G][r] = all[G].col[r]; t.ph[G][r] = all[G].ph[r]; }
}

int launch_contract(tsm_ctx* ctx, int slot)
{
    const Geom& g = ctx->g;
    const int nrhs = ctx->slot_nrhs[slot], prec = ctx->slot_prec[slot];
    int nblk = (g.Vsh + CT_BS - 1) / CT_BS;
    if (nblk > CT_MAXBLK) nblk = CT_MAXBLK;
    const size_t need = (size_t)nrhs * CT_NGROUP * g.L[3] * 2 * nblk * 32;
    if (need > ctx->partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const uint32_t* ids = ctx->ids_dev + slot * TSM_MAX_NRHS;
    const uint64_t seed = ctx->slot_seed[slot];
    const int kind = ctx->slot_kind[slot];
    const dim3 grid_l(nblk, g.L[3], nrhs * 2), grid_d(nblk * 4, g.L[3], nrhs * 2), grid_m(nblk * (ctx->n_mom > 0 ? ctx->n_mom : 1), g.L[3], nrhs * 2);
    Momenta mom;
    for (int m = 0; m < TSM_MAX_MOMENTA; m++)
        for (int k = 0; k < 3; k++) mom.n[m][k] = m < ctx->n_mom ? ctx->mom[m][k] : 0;
    const void* sol = ctx->slot[slot];
    // N2: second = D_W s = (1 - kappa D_hop) s on the full lattice, into the (idle) solver vectors
    void* second = ctx->vec[0];
    if (ctx->with_gen_one_end) {
        if (!ctx->have_params) return tsm_fail(ctx, TSM_ESTATE, "generalised one-end loops need kappa (tsm_set_params)");
        const size_t fp = field_bytes(prec, g.Vh, nrhs);
        const TwistCoef one = {1, 0, 1, 0}, mk = {-ctx->kappa, 0, -ctx->kappa, 0};
        const char* s_e = (const char*)sol; const char* s_o = s_e + fp;
        int rc;
        if ((rc = launch_dslash(ctx, prec, 0, false, nrhs, s_o, s_e, second, {one, mk}, 0))) return rc;
        if ((rc = launch_dslash(ctx, prec, 1, false, nrhs, s_e, s_o, (char*)second + fp, {one, mk}, 0))) return rc;
    }
#define CT(P, R)                                                                                                             \
    do {                                                                                                                     \
        const void* p0 = (P == TSM_F64) ? ctx->gauge64[0] : ctx->gauge32[0];                                                 \
        const void* p1 = (P == TSM_F64) ? ctx->gauge64[1] : ctx->gauge32[1];                                                 \
        int pi = prof_begin(ctx, P, 5, nrhs);                                                                                \
        k_contract<P, R, CT_LOCAL><<<grid_l, CT_BS, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials, mom); \
        prof_end(ctx, pi);                                                                                                   \
        ctx->launches++;                                                                                                     \
        if (ctx->with_deriv) {                                                                                               \
            pi = prof_begin(ctx, P, 6, nrhs);                                                                                \
            k_contract<P, R, CT_DERIV><<<grid_d, CT_BS, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials, mom); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
        if (ctx->with_momenta && ctx->n_mom > 0) {                                                                           \
            pi = prof_begin(ctx, P, 9, nrhs);                                                                                \
            k_contract<P, R, CT_MOMENTUM><<<grid_m, CT_BS, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials, mom); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
        if (ctx->with_gen_one_end) {                                                                                         \
            pi = prof_begin(ctx, P, 8, nrhs);                                                                                \
            k_contract<P, R, CT_GEN_ONE_END><<<grid_l, CT_BS, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials, mom); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
        if (ctx->with_one_end) {                                                                                             \
            pi = prof_begin(ctx, P, 7, nrhs);                                                                                \
            k_contract<P, R, CT_ONE_END><<<grid_l, CT_BS, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials, mom); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
    } while (0)
    if (prec == TSM_F64) CT(TSM_F64, 18);
    else if (prec == TSM_F32 && ctx->recon == 18) CT(TSM_F32, 18);
    else if (prec == TSM_F32) CT(TSM_F32, 12);
    else return tsm_fail(ctx, TSM_ESTATE, "slot holds no fp64/fp32 solution");
#undef CT
    TSM_CUDA(ctx, cudaGetLastError());
    OpBase ob;
    ob.v[0] = 0;
    for (int m = 0; m < 4; m++) ob.v[1 + m] = ctx->with_deriv ? TSM_N_LOCAL_OPS + 16 * m : -1;
    ob.v[5] = ctx->with_one_end ? TSM_N_LOCAL_OPS + (ctx->with_deriv ? TSM_N_DERIV_OPS : 0) : -1;
    ob.v[6] = ctx->with_gen_one_end ? TSM_N_LOCAL_OPS + (ctx->with_deriv ? TSM_N_DERIV_OPS : 0) + (ctx->with_one_end ? TSM_N_ONE_END_OPS : 0) : -1;
    {
        const int base = TSM_N_LOCAL_OPS + (ctx->with_deriv ? TSM_N_DERIV_OPS : 0) + (ctx->with_one_end ? TSM_N_ONE_END_OPS : 0) +
                         (ctx->with_gen_one_end ? TSM_N_GEN_ONE_END_OPS : 0);
        for (int m = 0; m < TSM_MAX_MOMENTA; m++) ob.v[7 + m] = (ctx->with_momenta && m < ctx->n_mom) ? base + 16 * m : -1;
    }
    if (ctx->with_one_end && !ctx->have_params) return tsm_fail(ctx, TSM_ESTATE, "one-end loops need kappa/mu (tsm_set_params)");
    const dim3 grid_f(g.L[3], CT_NGROUP, nrhs);
    k_contract_finish<<<grid_f, 32, 0, ctx->stream>>>(g.L[3], nblk, ctx->n_ops, ctx->gam, ob, 2.0 * (2.0 * ctx->kappa * ctx->mu),
                                                      ctx->partials, ctx->loops_src[slot]);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_accumulate(tsm_ctx* ctx, double* acc, const double* a, const double* b, int nrhs)
{
    const int n = ctx->n_ops * ctx->g.L[3] * 2;
    k_accumulate<<<(n + 255) / 256, 256, 0, ctx->stream>>>(n, nrhs, acc, a, b);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_finalize(tsm_ctx* ctx)
{
    const int n = ctx->n_ops * ctx->g.L[3] * 2;
    const double w_hp = ctx->n_hp > 0 ? 1.0 / ctx->n_hp : 0.0, w_lp = ctx->n_lp > 0 ? 1.0 / ctx->n_lp : 0.0;
    k_finalize<<<(n + 255) / 256, 256, 0, ctx->stream>>>(n, ctx->acc_corr, ctx->acc_lp, w_hp, w_lp, ctx->loops_out);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}
