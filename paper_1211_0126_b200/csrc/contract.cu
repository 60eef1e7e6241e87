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
#include "dslash_common.cuh"
#include "reduce.cuh"

namespace {

constexpr int CT_MAXBLK = 8;   // blocks per (timeslice, parity)
constexpr int CT_SPB = 8;      // sources (= warps) per block at most

// partials: [rhs][group][t][par][blk][32], group 0 local, 1..4 derivative mu, 5 one-end, 6 generalised one-end,
// 7 + m momentum m
constexpr int CT_NGROUP = 7 + TSM_MAX_MOMENTA;
enum { CT_LOCAL = 0, CT_DERIV = 1, CT_ONE_END = 2, CT_GEN_ONE_END = 3 };
struct Momenta { int n[TSM_MAX_MOMENTA][3]; };

// Transposed butterfly: every lane brings 32 values v[0..31]; lane L returns sum over the warp's lanes of THEIR
// v[L].  31 shuffles per lane instead of 32 x 5 for 32 separate tree sums, and a fixed tree (A19).  v is destroyed.
template <typename T> __device__ __forceinline__ T warp_transpose_sum(T* v)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        const bool up = (lane & o) != 0;
#pragma unroll
        for (int i = 0; i < o; i++) {
            const T keep = up ? v[i + o] : v[i];
            const T send = up ? v[i] : v[i + o];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
        }
    }
    return v[0];
}

// d[2 (4 al + be) + ri] += conj(l_{al c}) r_{be c} summed over c: the 4 x 4 spin matrix of one site is ADDED to d, in
// the precision of the field (fp32: packed, two FFMA2 per term; the sums over many sites are taken in fp64 by the caller)
template <typename T> __device__ __forceinline__ void spin_matrix(const T* l, const T* r, T* d)
{
    if constexpr (sizeof(T) == 4) {
        f2 a[16];
#pragma unroll
        for (int k = 0; k < 16; k++) a[k] = pk(d[2 * k], d[2 * k + 1]);
#pragma unroll
        for (int al = 0; al < 4; al++)
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const float lr = l[2 * (3 * al + c)], li = l[2 * (3 * al + c) + 1];
#pragma unroll
                for (int be = 0; be < 4; be++) {
                    const float rr = r[2 * (3 * be + c)], ri = r[2 * (3 * be + c) + 1];
                    a[4 * al + be] = fma2(pk(rr, ri), bc(lr), a[4 * al + be]);       // + lr * r
                    a[4 * al + be] = fma2(c_mi(rr, ri), bc(li), a[4 * al + be]);     // + li * (-i r)
                }
            }
#pragma unroll
        for (int k = 0; k < 16; k++) upk(a[k], d[2 * k], d[2 * k + 1]);
    } else {
#pragma unroll
        for (int al = 0; al < 4; al++)
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const T lr = l[2 * (3 * al + c)], li = l[2 * (3 * al + c) + 1];
#pragma unroll
                for (int be = 0; be < 4; be++) {
                    const T rr = r[2 * (3 * be + c)], ri = r[2 * (3 * be + c) + 1];
                    d[2 * (4 * al + be)] += lr * rr + li * ri;
                    d[2 * (4 * al + be) + 1] += lr * ri - li * rr;
                }
            }
    }
}

// eta_q = i^k (Z4) or 1 - 2 (k & 1) (Z2), k = bits 2q, 2q+1 (O3), straight into IEEE bit patterns: the value is
// +-1 in the real (k even) or the imaginary (k odd) part, the sign is bit 1 of k (Z4) or bit 0 (Z2)
template <typename T> __device__ __forceinline__ void noise_spinor(uint32_t bits, int kind, T* eta)
{
    const int sign_bit = kind == TSM_Z4 ? 1 : 0;
    const uint32_t odd_mask = kind == TSM_Z4 ? 1u : 0u;
#pragma unroll
    for (int q = 0; q < 12; q++) {
        const uint32_t k = bits >> (2 * q);
        const uint32_t one = 0x3f800000u | (((k >> sign_bit) & 1u) << 31);   // +-1.0f
        const bool odd = (k & odd_mask) != 0;
        eta[2 * q] = (T)__uint_as_float(odd ? 0u : one);
        eta[2 * q + 1] = (T)__uint_as_float(odd ? one : 0u);
    }
}

// One warp = one source on 32 consecutive cb sites of one (timeslice, parity) at a time; the warps of a block are
// the sources of the batch on the SAME sites (their link loads meet in L1).  grid = (nblk, 2 Lt, ceil(nrhs /
// blockDim.y)).  Per site the 4 x 4 spin matrix is formed in the field's precision; a lane adds up the matrices of SPL
// sites (in that precision: at most 4 x 3 colour terms per entry), the 32 lanes' sums are combined by the transposed
// butterfly (lane L ends with entry L), and each lane adds its entry to an fp64 accumulator.
// MODE 0: local; 1: derivative, all four directions in one pass (eta, the site decoding and the neighbour table are
// made once; one fp64 accumulator per direction); 2: one-end; 3: generalised one-end (second = D_W s, same
// [parity][rhs] layout as sol).
template <int PREC, int RECON, int MODE>
__global__ void __launch_bounds__(32 * CT_SPB, PREC == TSM_F64 ? 1 : 2) k_contract(const Geom g, const int nrhs, const int nblk, const void* __restrict__ sol,
                                                          const void* __restrict__ second, const void* __restrict__ pack0,
                                                          const void* __restrict__ pack1, const uint64_t seed, const uint32_t* __restrict__ ids,
                                                          const int kind, double* __restrict__ partials)
{
    using T = typename PT<PREC>::real;
    constexpr int SPL = MODE == CT_DERIV ? 1 : 4;   // sites per lane between two butterflies
    constexpr int NACC = MODE == CT_DERIV ? 4 : 1;
    const int lane = threadIdx.x, rhs = blockIdx.z * blockDim.y + threadIdx.y;
    if (rhs >= nrhs) return;
    const int Vh = g.Vh;
    const int blk = blockIdx.x;
    const int t = blockIdx.y >> 1, par = blockIdx.y & 1;
    const size_t fpar = field_bytes(PREC, Vh, nrhs), frhs = field_bytes(PREC, Vh, 1);
    const char* s_same = (const char*)sol + fpar * par + frhs * rhs;
    const char* s_other = (const char*)sol + fpar * (1 - par) + frhs * rhs;
    const void* pack = par ? pack1 : pack0;
    const uint32_t sid = ids[rhs];
    const int ngroup = (g.Vsh + 32 * SPL - 1) / (32 * SPL);
    double acc[NACC];
#pragma unroll
    for (int m = 0; m < NACC; m++) acc[m] = 0.0;

    if constexpr (MODE == CT_DERIV) {
        for (int gi = blk; gi < ngroup; gi += nblk) {
            const int jj = gi * 32 + lane;
            const bool live = jj < g.Vsh;
            const int i = t * g.Vsh + (live ? jj : 0);
            const SiteCoord sc = decode_site(g, i, par);
            T l[24];
            int nb[8];
            noise_spinor(noise_bits(lex_of_site(g, sc), seed, sid, kind), kind, l);
            neighbours(g, i, sc, nb);
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                T d[32];
#pragma unroll
                for (int k = 0; k < 32; k++) d[k] = 0;
                if (live) {
                    T uf[18], ub[18], sf[24], sb[24], a[6], b[6], r[24];
                    load_link_pair<PREC, RECON>(pack, i, mu, uf, ub);
                    load_spinor<PREC>(s_other, nb[2 * mu], sf);
                    load_spinor<PREC>(s_other, nb[2 * mu + 1], sb);
                    const T hf = (mu == 3 && sc.t == g.L[3] - 1) ? (T)0.5 * (T)g.theta : (T)0.5;
                    const T hb = (mu == 3 && sc.t == 0) ? (T)-0.5 * (T)g.theta : (T)-0.5;
#pragma unroll
                    for (int al = 0; al < 4; al++) {
                        su3_mul(uf, sf + 6 * al, a);
                        su3_mul(ub, sb + 6 * al, b);
#pragma unroll
                        for (int k = 0; k < 6; k++) r[6 * al + k] = hf * a[k] + hb * b[k];   // (D_mu s)(x), O6b
                    }
                    spin_matrix(l, r, d);
                }
                acc[mu] += (double)warp_transpose_sum(d);
            }
        }
    } else {
        for (int gi = blk; gi < ngroup; gi += nblk) {
            T dsum[32];
#pragma unroll
            for (int k = 0; k < 32; k++) dsum[k] = 0;
#pragma unroll
            for (int u = 0; u < SPL; u++) {
                const int jj = (gi * SPL + u) * 32 + lane;
                if (jj < g.Vsh) {
                    const int i = t * g.Vsh + jj;
                    T l[24], r[24];
                    if (MODE == CT_LOCAL) noise_spinor(noise_bits(lex_of_site(g, decode_site(g, i, par)), seed, sid, kind), kind, l);
                    if (MODE == CT_GEN_ONE_END) {
                        load_spinor<PREC>(s_same, i, l);
                        load_spinor<PREC>((const char*)second + fpar * par + frhs * rhs, i, r);
                    } else {
                        load_spinor<PREC>(s_same, i, r);
                        if (MODE == CT_ONE_END) {
#pragma unroll
                            for (int k = 0; k < 24; k++) l[k] = r[k];
                        }
                    }
                    spin_matrix(l, r, dsum);
                }
            }
            acc[0] += (double)warp_transpose_sum(dsum);
        }
    }
#pragma unroll
    for (int m = 0; m < NACC; m++) {
        const int group = MODE == CT_DERIV ? 1 + m : (MODE == CT_ONE_END ? 5 : (MODE == CT_GEN_ONE_END ? 6 : 0));
        const size_t o = ((((size_t)rhs * CT_NGROUP + group) * g.L[3] + t) * 2 + par) * nblk + blk;
        partials[o * 32 + lane] = acc[m];
    }
}

// N3: the same for the momentum-projected local loops, all momenta in ONE pass over s: the site's spin matrix is
// multiplied by each momentum's phase exp(2 pi i n.x/L) (product of three tabulated 1-d phases) before the butterfly;
// lane L keeps entry L of every momentum's sum in fp64.  Dynamic shared memory: the phase tables [nmom][Lx+Ly+Lz].
template <int PREC, int NM>   // NM: compile-time bound on nmom (8 or 16)
__global__ void __launch_bounds__(32 * CT_SPB) k_contract_momenta(const Geom g, const int nrhs, const int nblk, const int nmom,
                                                                  const void* __restrict__ sol, const uint64_t seed,
                                                                  const uint32_t* __restrict__ ids, const int kind,
                                                                  double* __restrict__ partials, const Momenta mom)
{
    using T = typename PT<PREC>::real;
    extern __shared__ __align__(16) double2 cm_smem[];
    double2* TB = cm_smem;   // [nmom][Lx + Ly + Lz]: exp(2 pi i n_d k / L_d), k = 0..L_d-1
    const int nl = g.L[0] + g.L[1] + g.L[2];
    for (int o = threadIdx.y * 32 + threadIdx.x; o < nmom * nl; o += 32 * blockDim.y) {
        const int m = o / nl, k = o - m * nl;
        const int dd = k < g.L[0] ? 0 : (k < g.L[0] + g.L[1] ? 1 : 2);
        const int kk = k - (dd == 0 ? 0 : (dd == 1 ? g.L[0] : g.L[0] + g.L[1])), L = g.L[dd];
        const int n = ((mom.n[m][dd] % L) + L) % L;             // the fraction n k / L reduced in integers first
        double sn, cs;
        sincospi(2.0 * (double)((n * kk) % L) / (double)L, &sn, &cs);
        TB[o] = make_double2(cs, sn);
    }
    __syncthreads();
    const int lane = threadIdx.x, rhs = blockIdx.z * blockDim.y + threadIdx.y;
    if (rhs >= nrhs) return;
    const int Vh = g.Vh, blk = blockIdx.x, t = blockIdx.y >> 1, par = blockIdx.y & 1;
    const char* s_same = (const char*)sol + field_bytes(PREC, Vh, nrhs) * par + field_bytes(PREC, Vh, 1) * rhs;
    const uint32_t sid = ids[rhs];
    const int nchunk = (g.Vsh + 31) >> 5;
    double acc[NM];
#pragma unroll
    for (int m = 0; m < NM; m++) acc[m] = 0.0;

    for (int ch = blk; ch < nchunk; ch += nblk) {
        const int jj = ch * 32 + lane;
        const bool live = jj < g.Vsh;
        const int i = t * g.Vsh + (live ? jj : 0);
        T d[32];
#pragma unroll
        for (int k = 0; k < 32; k++) d[k] = 0;
        SiteCoord sc = decode_site(g, i, par);
        if (live) {
            T l[24], r[24];
            noise_spinor(noise_bits(lex_of_site(g, sc), seed, sid, kind), kind, l);
            load_spinor<PREC>(s_same, i, r);
            spin_matrix(l, r, d);
        }
        const int x = 2 * sc.xh + sc.rowpar;
#pragma unroll
        for (int m = 0; m < NM; m++) {
            if (m < nmom) {   // warp-uniform
                const double2 a = TB[m * nl + x], b = TB[m * nl + g.L[0] + sc.y], c = TB[m * nl + g.L[0] + g.L[1] + sc.z];
                const double abr = a.x * b.x - a.y * b.y, abi = a.x * b.y + a.y * b.x;
                const T pr = (T)(abr * c.x - abi * c.y), pi = (T)(abr * c.y + abi * c.x);
                T wv[32];
                if constexpr (sizeof(T) == 4) cscale_f32<16>(pr, pi, d, wv);
                else {
#pragma unroll
                    for (int k = 0; k < 16; k++) {
                        wv[2 * k] = pr * d[2 * k] - pi * d[2 * k + 1];
                        wv[2 * k + 1] = pr * d[2 * k + 1] + pi * d[2 * k];
                    }
                }
                acc[m] += (double)warp_transpose_sum(wv);
            }
        }
    }
#pragma unroll
    for (int m = 0; m < NM; m++)
        if (m < nmom) {
            const size_t ob = ((((size_t)rhs * CT_NGROUP + 7 + m) * g.L[3] + t) * 2 + par) * nblk + blk;
            partials[ob * 32 + lane] = acc[m];
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
    int nblk = (g.Vsh + 32 * 32 - 1) / (32 * 32);   // 32 chunks of 32 sites per warp where the timeslice allows
    if (nblk < 1) nblk = 1;
    if (nblk > CT_MAXBLK) nblk = CT_MAXBLK;
    const int spb = nrhs < CT_SPB ? nrhs : CT_SPB;        // sources (warps) per block
    const int gz = (nrhs + spb - 1) / spb;
    const dim3 cblock(32, spb);
    const size_t need = (size_t)nrhs * CT_NGROUP * g.L[3] * 2 * nblk * 32;
    if (need > ctx->partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    const uint32_t* ids = ctx->ids_dev + slot * TSM_MAX_NRHS;
    const uint64_t seed = ctx->slot_seed[slot];
    const int kind = ctx->slot_kind[slot];
    const dim3 grid_l(nblk, 2 * g.L[3], gz), grid_d = grid_l;
    const size_t cm_smem_bytes = (size_t)(ctx->n_mom > 0 ? ctx->n_mom : 1) * (g.L[0] + g.L[1] + g.L[2]) * sizeof(double2);
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
        k_contract<P, R, CT_LOCAL><<<grid_l, cblock, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials); \
        prof_end(ctx, pi);                                                                                                   \
        ctx->launches++;                                                                                                     \
        if (ctx->with_deriv) {                                                                                               \
            pi = prof_begin(ctx, P, 6, nrhs);                                                                                \
            k_contract<P, R, CT_DERIV><<<grid_d, cblock, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
        if (ctx->with_momenta && ctx->n_mom > 0) {                                                                           \
            pi = prof_begin(ctx, P, 9, nrhs);                                                                                \
            if (ctx->n_mom <= 8)                                                                                             \
                k_contract_momenta<P, 8><<<grid_l, cblock, cm_smem_bytes, ctx->stream>>>(g, nrhs, nblk, ctx->n_mom, sol, seed, ids, kind, ctx->partials, mom); \
            else                                                                                                             \
                k_contract_momenta<P, 16><<<grid_l, cblock, cm_smem_bytes, ctx->stream>>>(g, nrhs, nblk, ctx->n_mom, sol, seed, ids, kind, ctx->partials, mom); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
        if (ctx->with_gen_one_end) {                                                                                         \
            pi = prof_begin(ctx, P, 8, nrhs);                                                                                \
            k_contract<P, R, CT_GEN_ONE_END><<<grid_l, cblock, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials); \
            prof_end(ctx, pi);                                                                                               \
            ctx->launches++;                                                                                                 \
        }                                                                                                                    \
        if (ctx->with_one_end) {                                                                                             \
            pi = prof_begin(ctx, P, 7, nrhs);                                                                                \
            k_contract<P, R, CT_ONE_END><<<grid_l, cblock, 0, ctx->stream>>>(g, nrhs, nblk, sol, second, p0, p1, seed, ids, kind, ctx->partials); \
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

// ------------------------------------------------------------------ the entry point that allocates nothing
// tsm_loops_local_noalloc (include/tsm.h): the local 16-Gamma loops (H8) of a caller-held solution field, for callers
// that cannot have device memory allocated on their behalf and have set no workspace.  It is the LOCAL mode of
// k_contract with two differences: the source ids travel by value in the kernel arguments (no id buffer), and the
// per-block partial sums go to g_na_scratch, a file-scope array of a fixed size that every GPU loading the library
// holds until exit, instead of the workspace's reduction scratch.  Same per-site arithmetic, same butterfly, same
// order over blocks in the finish kernel: the result is bit-identical to tsm_loops_source's local loops.
// Every call uses the same array: two calls that overlap on the GPU (different streams) race; calls on one stream are
// ordered.  Nothing in it has to start at zero: each call overwrites every entry its finish kernel reads.
constexpr size_t NA_MAX_DOUBLES = 524288;   // 4 MiB: nrhs * Lt * 2 * nblk * 32 doubles (32^3 x 64 with 16 sources fits exactly)
static __device__ __align__(256) double g_na_scratch[NA_MAX_DOUBLES];

namespace {

struct NaIds { uint32_t v[TSM_MAX_NRHS]; };

// scratch: [rhs][t][par][blk][32]
template <int PREC>
__global__ void __launch_bounds__(32 * CT_SPB, PREC == TSM_F64 ? 1 : 2) k_contract_local_na(const Geom g, const int nrhs, const int nblk, const void* __restrict__ sol,
                                                                   const uint64_t seed, const NaIds ids, const int kind, double* __restrict__ scratch)
{
    using T = typename PT<PREC>::real;
    constexpr int SPL = 4;   // sites per lane between two butterflies, as in k_contract
    const int lane = threadIdx.x, rhs = blockIdx.z * blockDim.y + threadIdx.y;
    if (rhs >= nrhs) return;
    const int Vh = g.Vh, blk = blockIdx.x, t = blockIdx.y >> 1, par = blockIdx.y & 1;
    const char* s_same = (const char*)sol + field_bytes(PREC, Vh, nrhs) * par + field_bytes(PREC, Vh, 1) * rhs;
    const uint32_t sid = ids.v[rhs];
    const int ngroup = (g.Vsh + 32 * SPL - 1) / (32 * SPL);
    double acc = 0.0;
    for (int gi = blk; gi < ngroup; gi += nblk) {
        T dsum[32];
#pragma unroll
        for (int k = 0; k < 32; k++) dsum[k] = 0;
#pragma unroll
        for (int u = 0; u < SPL; u++) {
            const int jj = (gi * SPL + u) * 32 + lane;
            if (jj < g.Vsh) {
                const int i = t * g.Vsh + jj;
                T l[24], r[24];
                noise_spinor(noise_bits(lex_of_site(g, decode_site(g, i, par)), seed, sid, kind), kind, l);
                load_spinor<PREC>(s_same, i, r);
                spin_matrix(l, r, dsum);
            }
        }
        acc += (double)warp_transpose_sum(dsum);
    }
    scratch[(((((size_t)rhs * g.L[3] + t) * 2 + par) * nblk + blk) << 5) + lane] = acc;
}

// grid = (Lt, nrhs), 32 threads: sums the blocks' partials in k_contract_finish's order and applies the 16 Gamma
__global__ void k_contract_finish_na(const int Lt, const int nblk, const GammaTable gt, const double* __restrict__ scratch, double* __restrict__ loops)
{
    const int t = blockIdx.x, rhs = blockIdx.y, k = threadIdx.x;
    __shared__ double C[32];
    double tot = 0;
    for (int pb = 0; pb < 2 * nblk; pb++) tot += scratch[((((size_t)rhs * Lt + t) * 2 * nblk + pb) << 5) + k];
    C[k] = tot;
    __syncthreads();
    if (k < 16) {
        double re = 0, im = 0;
        for (int al = 0; al < 4; al++) {
            const int be = gt.col[k][al], ph = gt.ph[k][al] & 3;
            const double cr = C[2 * (4 * al + be)], ci = C[2 * (4 * al + be) + 1];
            re += (ph == 0) ? cr : (ph == 1) ? -ci : (ph == 2) ? -cr : ci;   // times i^ph
            im += (ph == 0) ? ci : (ph == 1) ? cr : (ph == 2) ? -ci : -cr;
        }
        double* dst = loops + (((size_t)rhs * TSM_N_LOCAL_OPS + k) * Lt + t) * 2;
        dst[0] = re;
        dst[1] = im;
    }
}

}  // namespace

extern "C" size_t tsm_noalloc_scratch_bytes(void) { return NA_MAX_DOUBLES * sizeof(double); }

extern "C" int tsm_loops_local_noalloc(tsm_ctx* ctx, int prec, int nrhs, const void* dev_solution, uint64_t seed, const uint32_t* source_ids,
                                       int kind, double* dev_loops)
{
    int rc = ctx_enter(ctx, false, false, false);   // cudaSetDevice(ctx->device); needs no workspace, gauge field or parameters
    if (rc) return rc;
    if (!dev_solution || !dev_loops || !source_ids || nrhs < 1 || nrhs > TSM_MAX_NRHS || (prec != TSM_F64 && prec != TSM_F32) ||
        (kind != TSM_Z4 && kind != TSM_Z2))
        return tsm_fail(ctx, TSM_EINVAL, "bad no-alloc contraction arguments (prec must be TSM_F64 or TSM_F32, 1 <= nrhs <= 16)");
    const Geom& g = ctx->g;
    int nblk = (g.Vsh + 32 * 32 - 1) / (32 * 32);   // as launch_contract: the same blocks, hence the same sums
    if (nblk < 1) nblk = 1;
    if (nblk > CT_MAXBLK) nblk = CT_MAXBLK;
    const size_t need = (size_t)nrhs * g.L[3] * 2 * nblk * 32;
    if (need > NA_MAX_DOUBLES)
        return tsm_fail(ctx, TSM_EINVAL, "no-alloc contraction: nrhs * Lt * 2 * nblk * 32 doubles exceed the 4 MiB static scratch "
                                         "(tsm_noalloc_scratch_bytes); use fewer sources per call or tsm_loops_source");
    // The array's name is a host-side stand-in in host code: its device address is looked up once per device, with that
    // device current (ctx_enter has just made it so), and handed to the kernels.
    static double* scratch_of_device[64] = {nullptr};
    if (ctx->device >= 64) return tsm_fail(ctx, TSM_EINVAL, "no-alloc contraction: device index beyond 63");
    if (!scratch_of_device[ctx->device]) {
        void* p = nullptr;
        TSM_CUDA(ctx, cudaGetSymbolAddress(&p, g_na_scratch));
        if (!p) return tsm_fail(ctx, TSM_ECUDA, "cudaGetSymbolAddress returned no address for the static scratch");
        scratch_of_device[ctx->device] = (double*)p;
    }
    double* scratch = scratch_of_device[ctx->device];
    NaIds ids;
    for (int j = 0; j < TSM_MAX_NRHS; j++) ids.v[j] = j < nrhs ? source_ids[j] : 0u;
    const int spb = nrhs < CT_SPB ? nrhs : CT_SPB;
    const dim3 grid(nblk, 2 * g.L[3], (nrhs + spb - 1) / spb), block(32, spb);
    if (prec == TSM_F64) k_contract_local_na<TSM_F64><<<grid, block, 0, ctx->stream>>>(g, nrhs, nblk, dev_solution, seed, ids, kind, scratch);
    else k_contract_local_na<TSM_F32><<<grid, block, 0, ctx->stream>>>(g, nrhs, nblk, dev_solution, seed, ids, kind, scratch);
    k_contract_finish_na<<<dim3(g.L[3], nrhs), 32, 0, ctx->stream>>>(g.L[3], nblk, ctx->gam, scratch, dev_loops);
    ctx->launches += 2;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}
