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
//     a direct phase sum over a handful of momenta (not a full FFT), all momenta in one pass over s
//     (k_contract_momenta).
// H10 Eq. 2.4 accumulators (O7).
#include "reduce.cuh"

namespace {

constexpr int CT_BS = 128;
constexpr int CT_MAXBLK = 8;   // blocks per (timeslice, parity)

// grid = (nblk * ngroup_in_launch, Lt, nrhs * 2); MODE 0: local; 1: derivative, mu = blockIdx.x / nblk; 2: one-end;
// 3: generalised one-end (second = D_W s, same [parity][rhs] layout as sol).
// (the momentum-projected loops have their own kernel, k_contract_momenta)
// partials: [rhs][group][t][par][blk][32], group 0 local, 1..4 derivative mu, 5 one-end, 6 generalised one-end,
// 7 + m momentum m
constexpr int CT_NGROUP = 7 + TSM_MAX_MOMENTA;
enum { CT_LOCAL = 0, CT_DERIV = 1, CT_ONE_END = 2, CT_GEN_ONE_END = 3 };
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
        if (MODE == CT_LOCAL || MODE == CT_DERIV) bits = noise_bits(lex_of_site(g, sc), seed, sid, kind);
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
        const int group = MODE == CT_DERIV ? 1 + mu : (MODE == CT_ONE_END ? 5 : (MODE == CT_GEN_ONE_END ? 6 : 0));
        const size_t o = ((((size_t)rhs * CT_NGROUP + group) * g.L[3] + t) * 2 + par) * nblk + blk;
        partials[o * 32 + threadIdx.x] = tot;
    }
}

// N3 in ONE pass over s for all momenta.  grid = (nblk, Lt, nrhs * 2), 256 threads, dynamic shared memory.
// Per batch of 256 sites of the timeslice: (A) thread = site: regenerate eta, read s once, leave the site's 16
// complex d_{ab} = sum_c conj(eta_ac) s_bc in D[site][(ab + site) & 15] (swizzled: conflict-free both ways) and its
// nmom phases exp(2 pi i n.x/L) in P[m][site]; (B) thread = (entry ab, site lane sl): for its 16 sites of the
// batch, acc[m] += P[m][site] * D[site][ab] for every m (one D read serves all momenta).  At the end the 16 site
// lanes of an entry are summed in a fixed order and written where k_contract_finish expects group 7 + m.
constexpr int CM_BS = 256;
template <int PREC, int NM>   // NM: compile-time bound on nmom (8 or 16): the accumulators live in registers
__global__ void __launch_bounds__(CM_BS, NM <= 8 ? 2 : 1) k_contract_momenta(const Geom g, const int nrhs, const int nblk, const int nmom,
                                                            const void* __restrict__ sol, const uint64_t seed,
                                                            const uint32_t* __restrict__ ids, const int kind,
                                                            double* __restrict__ partials, const Momenta mom)
{
    using T = typename PT<PREC>::real;
    extern __shared__ __align__(16) double2 cm_smem[];
    double2* D = cm_smem;                       // [256 sites][16 entries]
    double2* P = cm_smem + CM_BS * 16;          // [nmom][256 sites]
    const int nl = g.L[0] + g.L[1] + g.L[2];
    double2* TB = P + nmom * CM_BS;             // [nmom][Lx + Ly + Lz]: exp(2 pi i n_d k / L_d), k = 0..L_d-1
    for (int o = threadIdx.x; o < nmom * nl; o += CM_BS) {
        const int m = o / nl, k = o - m * nl;
        const int d = k < g.L[0] ? 0 : (k < g.L[0] + g.L[1] ? 1 : 2);
        const int kk = k - (d == 0 ? 0 : (d == 1 ? g.L[0] : g.L[0] + g.L[1])), L = g.L[d];
        const int n = ((mom.n[m][d] % L) + L) % L;             // the fraction n k / L reduced in integers first
        double sn, cs;
        sincospi(2.0 * (double)((n * kk) % L) / (double)L, &sn, &cs);
        TB[o] = make_double2(cs, sn);
    }
    __syncthreads();
    const int Vh = g.Vh, tid = threadIdx.x;
    const int blk = blockIdx.x, t = blockIdx.y, rhs = blockIdx.z >> 1, par = blockIdx.z & 1;
    const char* s_same = (const char*)sol + field_bytes(PREC, Vh, nrhs) * par + field_bytes(PREC, Vh, 1) * rhs;
    const uint32_t sid = ids[rhs];
    const int e = tid & 15, sl = tid >> 4;
    double2 acc[NM];
#pragma unroll
    for (int m = 0; m < NM; m++) acc[m] = make_double2(0.0, 0.0);

    for (int base = blk * CM_BS; base < g.Vsh; base += nblk * CM_BS) {
        {   // (A)
            const int j = base + tid;
            double d[32];
#pragma unroll
            for (int k = 0; k < 32; k++) d[k] = 0.0;
            if (j < g.Vsh) {
                const int i = t * g.Vsh + j;
                const SiteCoord sc = decode_site(g, i, par);
                const uint32_t bits = noise_bits(lex_of_site(g, sc), seed, sid, kind);
                T v[24];
                load_spinor<PREC>(s_same, i, v);
#pragma unroll
                for (int al = 0; al < 4; al++)
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        float er, ei;
                        noise_value((bits >> (2 * (3 * al + c))) & 3, kind, er, ei);
                        const double cr = er, ci = -ei;   // conj(eta)
#pragma unroll
                        for (int be = 0; be < 4; be++) {
                            const double sr = (double)v[2 * (3 * be + c)], si = (double)v[2 * (3 * be + c) + 1];
                            d[2 * (4 * al + be)] += cr * sr - ci * si;
                            d[2 * (4 * al + be) + 1] += cr * si + ci * sr;
                        }
                    }
                const int x = 2 * sc.xh + sc.rowpar;
                for (int m = 0; m < nmom; m++) {   // exp(2 pi i n.x/L) as the product of the three tabulated 1-d phases
                    const double2 a = TB[m * nl + x], b = TB[m * nl + g.L[0] + sc.y], c = TB[m * nl + g.L[0] + g.L[1] + sc.z];
                    const double abr = a.x * b.x - a.y * b.y, abi = a.x * b.y + a.y * b.x;
                    P[m * CM_BS + tid] = make_double2(abr * c.x - abi * c.y, abr * c.y + abi * c.x);
                }
            } else {
                for (int m = 0; m < nmom; m++) P[m * CM_BS + tid] = make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int k = 0; k < 16; k++) D[tid * 16 + ((k + tid) & 15)] = make_double2(d[2 * k], d[2 * k + 1]);
        }
        __syncthreads();
        // (B)
#pragma unroll 4
        for (int q = 0; q < 16; q++) {
            const int site = sl + 16 * q;
            const double2 dv = D[site * 16 + ((e + site) & 15)];
#pragma unroll
            for (int m = 0; m < NM; m++) {
                if (m < nmom) {
                    const double2 ph = P[m * CM_BS + site];
                    acc[m].x += ph.x * dv.x - ph.y * dv.y;
                    acc[m].y += ph.x * dv.y + ph.y * dv.x;
                }
            }
        }
        __syncthreads();
    }
    // sum over the 16 site lanes of each entry, fixed order (A19); R[m][sl][e] reuses D
    double2* R = D;
#pragma unroll
    for (int m = 0; m < NM; m++)
        if (m < nmom) R[(m * 16 + sl) * 16 + e] = acc[m];
    __syncthreads();
    for (int o = tid; o < nmom * 16; o += CM_BS) {
        const int m = o >> 4, ee = o & 15;
        double re = 0, im = 0;
        for (int l = 0; l < 16; l++) { const double2 v = R[(m * 16 + l) * 16 + ee]; re += v.x; im += v.y; }
        const size_t ob = ((((size_t)rhs * CT_NGROUP + 7 + m) * g.L[3] + t) * 2 + par) * nblk + blk;
        partials[ob * 32 + 2 * ee] = re;
        partials[ob * 32 + 2 * ee + 1] = im;
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
    const dim3 grid_l(nblk, g.L[3], nrhs * 2), grid_d(nblk * 4, g.L[3], nrhs * 2);
    const size_t cm_smem_bytes = (size_t)CM_BS * 16 * sizeof(double2) +
                                 (size_t)(ctx->n_mom > 0 ? ctx->n_mom : 1) * (CM_BS + g.L[0] + g.L[1] + g.L[2]) * sizeof(double2);
    if (ctx->with_momenta && ctx->n_mom > 0) {
        TSM_CUDA(ctx, cudaFuncSetAttribute(k_contract_momenta<TSM_F64, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cm_smem_bytes));
        TSM_CUDA(ctx, cudaFuncSetAttribute(k_contract_momenta<TSM_F32, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cm_smem_bytes));
        TSM_CUDA(ctx, cudaFuncSetAttribute(k_contract_momenta<TSM_F64, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cm_smem_bytes));
        TSM_CUDA(ctx, cudaFuncSetAttribute(k_contract_momenta<TSM_F32, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cm_smem_bytes));
        if (cm_smem_bytes > 200 * 1024) return tsm_fail(ctx, TSM_EINVAL, "lattice too wide for the momentum phase tables");
    }
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
            if (ctx->n_mom <= 8)                                                                                             \
                k_contract_momenta<P, 8><<<grid_l, CM_BS, cm_smem_bytes, ctx->stream>>>(g, nrhs, nblk, ctx->n_mom, sol, seed, ids, kind, ctx->partials, mom); \
            else                                                                                                             \
                k_contract_momenta<P, 16><<<grid_l, CM_BS, cm_smem_bytes, ctx->stream>>>(g, nrhs, nblk, ctx->n_mom, sol, seed, ids, kind, ctx->partials, mom); \
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
