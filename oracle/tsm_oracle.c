/*
 * tsm_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU oracle for the
 * truncated-solver-method (TSM) disconnected-loop hot path of arXiv:1211.0126.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this.  It shares no code, header, table or constant
 * generator with the CUDA path under paper_1211_0126_b200/csrc/.
 *
 * Every function cites the passage it follows: "PAPER.md:<line>" is the paper,
 * "Ox/Ax/Cx" are the readings of SURVEY.md section 8(c), restated in DESIGN.md.
 * There is no blocking, fusion or reordering beyond those statements.  The only
 * parallelism is an OpenMP `parallel for` over output sites of the hopping term
 * (each site is independent); all dot products and norms are plain serial sums
 * so that results do not depend on the thread count.
 *
 * Pins (tests/test_oracle_*.py): P1 gamma algebra, P2 free-field spectrum,
 * P3 gamma5-hermiticity / adjointness, P4 twisted-mass identities, P5 even-odd
 * algebra, P6 gauge covariance, P7 dense brute force, P8 estimator statistics,
 * P9 free-field loops, P10 one-end identity, P11 TSM algebra, P12 Philox known
 * answers, P13 CG Krylov optimality, P14 derivative, P15 delta-source stencil.
 * P16 one-end trick (Eq. 2.5) against dense M(mu)^-1 - M(-mu)^-1, P17 generalised one-end
 * trick (Eq. 2.6) against dense M(mu)^-1 + M(-mu)^-1, P18 momentum-projected loops against numpy's FFT.
 * Parity unpinned (defined only by the algorithm O5): the values of truncated LP
 * iterates beyond P13's Krylov-minimiser check.
 *
 * Conventions (C1, C2): site x=(x0,x1,x2,x3)=(x,y,z,t), lex = x0+L0*(x1+L1*(x2+L2*x3));
 * spinor psi[lex][alpha][c] (alpha=0..3 spin, c=0..2 colour), link U[mu][lex][c][c'],
 * (U psi)_{alpha c} = sum_c' U_{cc'} psi_{alpha c'}; complex numbers as (re,im) doubles.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define NS 4
#define NC 3
#define SPINOR (NS * NC)

/* ------------------------------------------------------------------------- */
/* C3: gamma matrices in the chiral, hermitian, Euclidean basis.             */
/* gamma_k = [[0, -i sigma_k], [i sigma_k, 0]] (k=0,1,2 <-> x,y,z),          */
/* gamma_3 = [[0,1],[1,0]], gamma5 = gamma_0 gamma_1 gamma_2 gamma_3.         */
/* ------------------------------------------------------------------------- */
static void mat4_mul(const cplx a[4][4], const cplx b[4][4], cplx out[4][4])
{
    cplx t[4][4];
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            cplx s = 0;
            for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
            t[i][j] = s;
        }
    memcpy(out, t, sizeof(t));
}

static void build_gamma(cplx g[5][4][4])
{
    const cplx sigma[3][2][2] = {
        {{0, 1}, {1, 0}},
        {{0, -I}, {I, 0}},
        {{1, 0}, {0, -1}},
    };
    memset(g, 0, 5 * 16 * sizeof(cplx));
    for (int k = 0; k < 3; k++)
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) {
                g[k][i][2 + j] = -I * sigma[k][i][j];
                g[k][2 + i][j] = I * sigma[k][i][j];
            }
    for (int i = 0; i < 2; i++) {
        g[3][i][2 + i] = 1;
        g[3][2 + i][i] = 1;
    }
    cplx t[4][4];
    mat4_mul(g[0], g[1], t);
    mat4_mul(t, g[2], t);
    mat4_mul(t, g[3], g[4]);
}

/* The 16 Gamma of C3 in output order: 0:1, 1:g5, 2-5:g_mu, 6-9:g5 g_mu,
 * 10-15: sigma_{mu nu} = (i/2)[g_mu, g_nu] for (mu nu) = 01,02,03,12,13,23.
 * out is [4][4][2] (row alpha, column beta, re/im). */
void oracle_gamma(int idx, double *out)
{
    cplx g[5][4][4], G[4][4];
    build_gamma(g);
    memset(G, 0, sizeof(G));
    if (idx == 0) {
        for (int i = 0; i < 4; i++) G[i][i] = 1;
    } else if (idx == 1) {
        memcpy(G, g[4], sizeof(G));
    } else if (idx >= 2 && idx <= 5) {
        memcpy(G, g[idx - 2], sizeof(G));
    } else if (idx >= 6 && idx <= 9) {
        mat4_mul(g[4], g[idx - 6], G);
    } else if (idx >= 10 && idx <= 15) {
        static const int pair[6][2] = {{0, 1}, {0, 2}, {0, 3}, {1, 2}, {1, 3}, {2, 3}};
        int m = pair[idx - 10][0], n = pair[idx - 10][1];
        cplx a[4][4], b[4][4];
        mat4_mul(g[m], g[n], a);
        mat4_mul(g[n], g[m], b);
        for (int i = 0; i < 4; i++)
            for (int j = 0; j < 4; j++) G[i][j] = 0.5 * I * (a[i][j] - b[i][j]);
    }
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            out[2 * (4 * i + j)] = creal(G[i][j]);
            out[2 * (4 * i + j) + 1] = cimag(G[i][j]);
        }
}

/* ------------------------------------------------------------------------- */
/* C1: geometry                                                               */
/* ------------------------------------------------------------------------- */
static inline long vol(const int L[4]) { return (long)L[0] * L[1] * L[2] * L[3]; }

static inline long lex_of(const int L[4], const int x[4])
{
    return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3]));
}

static inline void coords_of(const int L[4], long lex, int x[4])
{
    x[0] = (int)(lex % L[0]); lex /= L[0];
    x[1] = (int)(lex % L[1]); lex /= L[1];
    x[2] = (int)(lex % L[2]); lex /= L[2];
    x[3] = (int)lex;
}

static inline int parity_of(const int x[4]) { return (x[0] + x[1] + x[2] + x[3]) & 1; }

/* ------------------------------------------------------------------------- */
/* O2: hopping term.  For every site x whose parity matches `par` (par<0: all)*/
/*   out(x) = sum_mu [ phi+_mu(x) U_mu(x) (1-g_mu) in(x+mu)                   */
/*                   + phi-_mu(x) U_mu(x-mu)^dag (1+g_mu) in(x-mu) ]          */
/* phi+_3(x)=theta if x3=Lt-1 else 1; phi-_3(x)=theta if x3=0 else 1;         */
/* spatial directions periodic.  Other-parity sites of `out` are set to 0.    */
/* (PAPER.md:58,64 fix M_u +- M_d; the Wilson form with r=1 is reading A1.)   */
/* ------------------------------------------------------------------------- */
void oracle_hop(const int L[4], int theta, const double *U_, const double *in_, double *out_, int par)
{
    const cplx *U = (const cplx *)U_;
    const cplx *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    const long V = vol(L);
    cplx g[5][4][4];
    build_gamma(g);

#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        int x[4];
        coords_of(L, s, x);
        cplx acc[NS][NC];
        memset(acc, 0, sizeof(acc));
        if (par < 0 || parity_of(x) == par) {
            for (int mu = 0; mu < 4; mu++) {
                int xp[4] = {x[0], x[1], x[2], x[3]}, xm[4] = {x[0], x[1], x[2], x[3]};
                xp[mu] = (x[mu] + 1) % L[mu];
                xm[mu] = (x[mu] + L[mu] - 1) % L[mu];
                const long sp = lex_of(L, xp), sm = lex_of(L, xm);
                const double phip = (mu == 3 && x[3] == L[3] - 1) ? (double)theta : 1.0;
                const double phim = (mu == 3 && x[3] == 0) ? (double)theta : 1.0;
                const cplx *Uf = U + ((long)mu * V + s) * 9;  /* U_mu(x)    */
                const cplx *Ub = U + ((long)mu * V + sm) * 9; /* U_mu(x-mu) */
                cplx tf[NS][NC], tb[NS][NC];
                for (int a = 0; a < NS; a++)
                    for (int c = 0; c < NC; c++) {
                        cplx f = 0, b = 0;
                        for (int bb = 0; bb < NS; bb++) {
                            const cplx d = (a == bb) ? 1.0 : 0.0;
                            f += (d - g[mu][a][bb]) * in[(sp * NS + bb) * NC + c];
                            b += (d + g[mu][a][bb]) * in[(sm * NS + bb) * NC + c];
                        }
                        tf[a][c] = f;
                        tb[a][c] = b;
                    }
                for (int a = 0; a < NS; a++)
                    for (int c = 0; c < NC; c++) {
                        cplx f = 0, b = 0;
                        for (int cc = 0; cc < NC; cc++) {
                            f += Uf[c * 3 + cc] * tf[a][cc];
                            b += conj(Ub[cc * 3 + c]) * tb[a][cc];
                        }
                        acc[a][c] += phip * f + phim * b;
                    }
            }
        }
        memcpy(out + s * SPINOR, acc, sizeof(acc));
    }
}

/* gamma5 psi, site by site (C3: gamma5 = g0 g1 g2 g3, used as a full matrix). */
static void apply_g5(long V, const cplx *in, cplx *out)
{
    cplx g[5][4][4];
    build_gamma(g);
    for (long s = 0; s < V; s++) {
        cplx t[NS][NC];
        for (int a = 0; a < NS; a++)
            for (int c = 0; c < NC; c++) {
                cplx v = 0;
                for (int b = 0; b < NS; b++) v += g[4][a][b] * in[(s * NS + b) * NC + c];
                t[a][c] = v;
            }
        memcpy(out + s * SPINOR, t, sizeof(t));
    }
}

/* O2: (M psi)(x) = psi(x) + i a gamma5 psi(x) - kappa hop(psi)(x), a = 2 kappa mu.
 * This is 2 kappa times the paper's M_u = D_W + i mu gamma5. */
void oracle_apply_M(const int L[4], int theta, double kappa, double mu, const double *U,
                    const double *in_, double *out_)
{
    const long V = vol(L);
    const double a = 2.0 * kappa * mu;
    const cplx *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    cplx *h = malloc(V * SPINOR * sizeof(cplx));
    cplx *g5 = malloc(V * SPINOR * sizeof(cplx));
    oracle_hop(L, theta, U, in_, (double *)h, -1);
    apply_g5(V, in, g5);
    for (long i = 0; i < V * SPINOR; i++) out[i] = in[i] + I * a * g5[i] - kappa * h[i];
    free(h);
    free(g5);
}

/* ------------------------------------------------------------------------- */
/* O4: even-odd preconditioning.  M = [[R, -kappa D_eo], [-kappa D_oe, R]],   */
/* R = 1 + i a gamma5, R^-1 = (1 - i a gamma5)/(1 + a^2).                     */
/* Fields are full-lattice arrays; the unused parity holds zeros.             */
/* ------------------------------------------------------------------------- */
static void apply_R(long V, double a, const cplx *in, cplx *out) /* out = (1 + i a g5) in */
{
    cplx *g5 = malloc(V * SPINOR * sizeof(cplx));
    apply_g5(V, in, g5);
    for (long i = 0; i < V * SPINOR; i++) out[i] = in[i] + I * a * g5[i];
    free(g5);
}

static void apply_Rinv(long V, double a, const cplx *in, cplx *out)
{
    cplx *g5 = malloc(V * SPINOR * sizeof(cplx));
    apply_g5(V, in, g5);
    for (long i = 0; i < V * SPINOR; i++) out[i] = (in[i] - I * a * g5[i]) / (1.0 + a * a);
    free(g5);
}

/* Mhat x = R x - kappa^2 D_eo R^-1 D_oe x on even sites (x zero on odd sites). */
static void apply_Mhat_a(const int L[4], int theta, double kappa, double a, const double *U,
                         const cplx *in, cplx *out)
{
    const long V = vol(L);
    cplx *t1 = malloc(V * SPINOR * sizeof(cplx));
    cplx *t2 = malloc(V * SPINOR * sizeof(cplx));
    oracle_hop(L, theta, U, (const double *)in, (double *)t1, 1); /* D_oe x : odd sites  */
    apply_Rinv(V, a, t1, t2);
    oracle_hop(L, theta, U, (const double *)t2, (double *)t1, 0); /* D_eo . : even sites */
    apply_R(V, a, in, t2);
    for (long i = 0; i < V * SPINOR; i++) out[i] = t2[i] - kappa * kappa * t1[i];
    free(t1);
    free(t2);
}

void oracle_apply_Mhat(const int L[4], int theta, double kappa, double mu, const double *U,
                       const double *in, double *out)
{
    apply_Mhat_a(L, theta, kappa, 2.0 * kappa * mu, U, (const cplx *)in, (cplx *)out);
}

/* Mhat^dagger = gamma5 Mhat(-mu) gamma5 (O4); pinned as the true adjoint by P3. */
void oracle_apply_Mhat_dag(const int L[4], int theta, double kappa, double mu, const double *U,
                           const double *in, double *out)
{
    const long V = vol(L);
    cplx *t = malloc(V * SPINOR * sizeof(cplx));
    apply_g5(V, (const cplx *)in, t);
    apply_Mhat_a(L, theta, kappa, -2.0 * kappa * mu, U, t, (cplx *)out);
    apply_g5(V, (const cplx *)out, (cplx *)out);
    free(t);
}

/* ------------------------------------------------------------------------- */
/* O3: Z4 / Z2 noise from Philox4x32-10 (Salmon et al., SC'11).               */
/* ------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; round++) {
        const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* eta(x, alpha, c) = i^k (Z4, kind 0) or 1-2(k&1) (Z2, kind 1), k = (word0 >> 2q) & 3,
 * q = 3 alpha + c, word0 the first output of Philox with key = (seed lo, seed hi),
 * counter = (lex lo, lex hi, source_id, 0x5A340000 | kind).  PAPER.md:28-30 ("each
 * component ... a particular representation of the Z2 or Z4 group"), readings A5, A6. */
void oracle_noise(const int L[4], uint64_t seed, uint32_t source_id, int kind, double *out_)
{
    cplx *out = (cplx *)out_;
    const long V = vol(L);
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    static const cplx z4[4] = {1, I, -1, -I};
    for (long s = 0; s < V; s++) {
        const uint32_t ctr[4] = {(uint32_t)((uint64_t)s & 0xffffffffu), (uint32_t)((uint64_t)s >> 32),
                                 source_id, 0x5A340000u | (uint32_t)kind};
        uint32_t w[4];
        oracle_philox4x32_10(ctr, key, w);
        for (int q = 0; q < SPINOR; q++) {
            const int k = (w[0] >> (2 * q)) & 3;
            out[s * SPINOR + q] = (kind == 0) ? z4[k] : (cplx)(1 - 2 * (k & 1));
        }
    }
}

/* ------------------------------------------------------------------------- */
/* O4 + O5: solve M s = eta by even-odd preconditioned CG on Mhat^dag Mhat.   */
/* PAPER.md:32 (solve M|s>=|eta>), :48 (truncation by residual or iteration   */
/* count), readings A7-A9, A13.                                               */
/* info[0]=iterations, info[1]=recursive relative residual sqrt(rr/|b'|^2),   */
/* info[2]=true relative residual |eta - M s|/|eta| of the full system,       */
/* info[3]=status (0 ok, -5 breakdown, -6 tolerance not reached in max_iter). */
/* ------------------------------------------------------------------------- */
static double norm2(long n, const cplx *v)
{
    double s = 0;
    for (long i = 0; i < n; i++) s += creal(v[i]) * creal(v[i]) + cimag(v[i]) * cimag(v[i]);
    return s;
}

static double re_dot(long n, const cplx *a, const cplx *b) /* Re <a,b> = Re sum conj(a) b */
{
    double s = 0;
    for (long i = 0; i < n; i++) s += creal(a[i]) * creal(b[i]) + cimag(a[i]) * cimag(b[i]);
    return s;
}

void oracle_solve(const int L[4], int theta, double kappa, double mu, const double *U,
                  const double *eta_, double tol, int max_iter, double *s_, double *info)
{
    const long V = vol(L), n = V * SPINOR;
    const double a = 2.0 * kappa * mu;
    const cplx *eta = (const cplx *)eta_;
    cplx *s = (cplx *)s_;
    cplx *eta_e = calloc(n, sizeof(cplx)), *eta_o = calloc(n, sizeof(cplx));
    cplx *t1 = malloc(n * sizeof(cplx)), *t2 = malloc(n * sizeof(cplx));
    cplx *bhat = malloc(n * sizeof(cplx)), *bp = malloc(n * sizeof(cplx));
    cplx *x = calloc(n, sizeof(cplx)), *r = malloc(n * sizeof(cplx)), *p = malloc(n * sizeof(cplx));
    cplx *w = malloc(n * sizeof(cplx)), *q = malloc(n * sizeof(cplx));

    for (long st = 0; st < V; st++) {
        int xx[4];
        coords_of(L, st, xx);
        cplx *dst = parity_of(xx) ? eta_o : eta_e;
        memcpy(dst + st * SPINOR, eta + st * SPINOR, SPINOR * sizeof(cplx));
    }
    /* O4: bhat = eta_e + kappa D_eo R^-1 eta_o */
    apply_Rinv(V, a, eta_o, t1);
    oracle_hop(L, theta, U, (const double *)t1, (double *)t2, 0);
    for (long i = 0; i < n; i++) bhat[i] = eta_e[i] + kappa * t2[i];
    /* O5: b' = Mhat^dag bhat, x0 = 0, r0 = p0 = b' */
    oracle_apply_Mhat_dag(L, theta, kappa, mu, U, (const double *)bhat, (double *)bp);
    memcpy(r, bp, n * sizeof(cplx));
    memcpy(p, bp, n * sizeof(cplx));
    const double bb = norm2(n, bp);
    double rr = bb;
    int iters = 0, status = 0;
    if (max_iter > 0 && bb > 0) {
        for (int k = 1;; k++) {
            oracle_apply_Mhat(L, theta, kappa, mu, U, (const double *)p, (double *)w);
            oracle_apply_Mhat_dag(L, theta, kappa, mu, U, (const double *)w, (double *)q);
            const double pq = re_dot(n, p, q);
            if (!(pq > 0) || !isfinite(pq) || !(rr > 0) || !isfinite(rr)) { /* A13 */
                status = -5;
                break;
            }
            const double alpha = rr / pq;
            for (long i = 0; i < n; i++) x[i] += alpha * p[i];
            for (long i = 0; i < n; i++) r[i] -= alpha * q[i];
            const double rr_new = norm2(n, r);
            iters = k;
            if (tol > 0 && sqrt(rr_new / bb) <= tol) { rr = rr_new; break; }
            if (k == max_iter) {
                rr = rr_new;
                if (tol > 0) status = -6;
                break;
            }
            const double beta = rr_new / rr;
            for (long i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
            rr = rr_new;
        }
    }
    /* O4: s_e = x, s_o = R^-1 (eta_o + kappa D_oe x) */
    oracle_hop(L, theta, U, (const double *)x, (double *)t1, 1);
    for (long i = 0; i < n; i++) t2[i] = eta_o[i] + kappa * t1[i];
    apply_Rinv(V, a, t2, t1);
    for (long i = 0; i < n; i++) s[i] = x[i] + t1[i];
    /* reading A8: the fp64 true residual of the full system is always reported */
    oracle_apply_M(L, theta, kappa, mu, U, (const double *)s, (double *)t1);
    for (long i = 0; i < n; i++) t1[i] = eta[i] - t1[i];
    info[0] = iters;
    info[1] = bb > 0 ? sqrt(rr / bb) : 0.0;
    info[2] = sqrt(norm2(n, t1) / norm2(n, eta));
    info[3] = status;
    free(eta_e); free(eta_o); free(t1); free(t2); free(bhat); free(bp);
    free(x); free(r); free(p); free(w); free(q);
}

/* True relative residual |eta - M s| / |eta| of any candidate solution (reading A17). */
double oracle_true_residual(const int L[4], int theta, double kappa, double mu, const double *U,
                            const double *eta, const double *s)
{
    const long n = vol(L) * SPINOR;
    cplx *t = malloc(n * sizeof(cplx));
    oracle_apply_M(L, theta, kappa, mu, U, s, (double *)t);
    for (long i = 0; i < n; i++) t[i] = ((const cplx *)eta)[i] - t[i];
    const double res = sqrt(norm2(n, t) / norm2(n, (const cplx *)eta));
    free(t);
    return res;
}

/* ------------------------------------------------------------------------- */
/* O6: local loops  L_Gamma(t) = sum_{x in t} sum_{alpha beta c}              */
/*        conj(eta_{alpha c}(x)) Gamma_{alpha beta} s_{beta c}(x)             */
/* PAPER.md:58 ((1/N) sum <eta^dag X s> ~ Tr(M^-1 X)), :84 (all insertion     */
/* times).  out is [16][Lt][2].                                               */
/* ------------------------------------------------------------------------- */
void oracle_loops(const int L[4], const double *eta_, const double *s_, double *out_)
{
    const cplx *eta = (const cplx *)eta_, *s = (const cplx *)s_;
    cplx *out = (cplx *)out_;
    const long V = vol(L), Vs = (long)L[0] * L[1] * L[2];
    const int T = L[3];
    for (int G = 0; G < 16; G++) {
        double gm[32];
        oracle_gamma(G, gm);
        for (int t = 0; t < T; t++) {
            cplx acc = 0;
            for (long sx = 0; sx < Vs; sx++) {
                const long st = (long)t * Vs + sx;
                for (int a = 0; a < NS; a++)
                    for (int b = 0; b < NS; b++) {
                        const cplx gab = gm[2 * (4 * a + b)] + I * gm[2 * (4 * a + b) + 1];
                        if (gab == 0) continue;
                        for (int c = 0; c < NC; c++)
                            acc += conj(eta[(st * NS + a) * NC + c]) * gab * s[(st * NS + b) * NC + c];
                    }
            }
            out[(long)G * T + t] = acc;
        }
    }
    (void)V;
}

/* O6b: (D_mu s)(x) = 1/2 [ phi+_mu(x) U_mu(x) s(x+mu) - phi-_mu(x) U_mu(x-mu)^dag s(x-mu) ]
 * (right-acting symmetric covariant difference, reading A18; PAPER.md:78 names the
 * operator i psibar gamma_3 D_3 psi).  out is [V][4][3] complex. */
void oracle_cov_diff(const int L[4], int theta, const double *U_, int mu, const double *s_, double *out_)
{
    const cplx *U = (const cplx *)U_, *s = (const cplx *)s_;
    cplx *out = (cplx *)out_;
    const long V = vol(L);
    for (long st = 0; st < V; st++) {
        int x[4];
        coords_of(L, st, x);
        int xp[4] = {x[0], x[1], x[2], x[3]}, xm[4] = {x[0], x[1], x[2], x[3]};
        xp[mu] = (x[mu] + 1) % L[mu];
        xm[mu] = (x[mu] + L[mu] - 1) % L[mu];
        const long sp = lex_of(L, xp), sm = lex_of(L, xm);
        const double phip = (mu == 3 && x[3] == L[3] - 1) ? (double)theta : 1.0;
        const double phim = (mu == 3 && x[3] == 0) ? (double)theta : 1.0;
        const cplx *Uf = U + ((long)mu * V + st) * 9, *Ub = U + ((long)mu * V + sm) * 9;
        for (int a = 0; a < NS; a++)
            for (int c = 0; c < NC; c++) {
                cplx f = 0, b = 0;
                for (int cc = 0; cc < NC; cc++) {
                    f += Uf[c * 3 + cc] * s[(sp * NS + a) * NC + cc];
                    b += conj(Ub[cc * 3 + c]) * s[(sm * NS + a) * NC + cc];
                }
                out[(st * NS + a) * NC + c] = 0.5 * (phip * f - phim * b);
            }
    }
}

/* O6b: L_{Gamma,mu}(t) = sum_{x in t} eta^dag(x) Gamma (D_mu s)(x); out is [4][16][Lt][2]. */
void oracle_loops_deriv(const int L[4], int theta, const double *U, const double *eta,
                        const double *s, double *out)
{
    const long V = vol(L);
    const int T = L[3];
    double *d = malloc(V * SPINOR * 2 * sizeof(double));
    for (int mu = 0; mu < 4; mu++) {
        oracle_cov_diff(L, theta, U, mu, s, d);
        oracle_loops(L, eta, d, out + (long)mu * 16 * T * 2);
    }
    free(d);
}

/* ------------------------------------------------------------------------- */
/* N1: the one-end trick, Eq. 2.5.             */
/*   (2 i mu a / N) sum_r <s_r gamma5 X s_r> = Tr(M_u^-1 X) - Tr(M_d^-1 X)    */
/* from M_u - M_d = 2 i mu a gamma5.  In the kappa-normalised   */
/* operator of O2 the identity reads M(mu) - M(-mu) = 2 i a gamma5, a = 2     */
/* kappa mu, and M(-mu) = gamma5 M(mu)^dag gamma5, hence                      */
/*   M_u^-1 - M_d^-1 = -2 i a M_u^-1 gamma5 M_d^-1,                           */
/*   E_eta[ s^dag gamma5 X s ] = Tr[X M_u^-1 gamma5 M_d^-1]  for s = M_u^-1 eta */
/* so the per-source, per-timeslice one-end loop whose noise average is       */
/* sum_{x in t} tr[Gamma (M_u^-1 - M_d^-1)(x,x)] is (reading A24: the sign is */
/* fixed by the right-hand side of Eq. 2.5 with s solving the mu > 0 flavour) */
/*   L1_Gamma(t; s) = -2 i a sum_{x in t} sum_{alpha beta c}                  */
/*                    conj(s_{alpha c}(x)) (gamma5 Gamma)_{alpha beta} s_{beta c}(x). */
/* out is [16][Lt][2].                                                        */
/* ------------------------------------------------------------------------- */
void oracle_loops_one_end(const int L[4], double kappa, double mu, const double *s_, double *out_)
{
    const cplx *s = (const cplx *)s_;
    cplx *out = (cplx *)out_;
    const long Vs = (long)L[0] * L[1] * L[2];
    const int T = L[3];
    const double a = 2.0 * kappa * mu;
    cplx g[5][4][4];
    build_gamma(g);
    for (int G = 0; G < 16; G++) {
        double gm[32];
        cplx Gam[4][4], g5G[4][4];
        oracle_gamma(G, gm);
        for (int i = 0; i < 4; i++)
            for (int j = 0; j < 4; j++) Gam[i][j] = gm[2 * (4 * i + j)] + I * gm[2 * (4 * i + j) + 1];
        mat4_mul(g[4], Gam, g5G);
        for (int t = 0; t < T; t++) {
            cplx acc = 0;
            for (long sx = 0; sx < Vs; sx++) {
                const long st = (long)t * Vs + sx;
                for (int al = 0; al < NS; al++)
                    for (int be = 0; be < NS; be++) {
                        if (g5G[al][be] == 0) continue;
                        for (int c = 0; c < NC; c++)
                            acc += conj(s[(st * NS + al) * NC + c]) * g5G[al][be] * s[(st * NS + be) * NC + c];
                    }
            }
            out[(long)G * T + t] = -2.0 * I * a * acc;
        }
    }
}

/* ------------------------------------------------------------------------- */
/* N2: the generalised one-end trick, Eq. 2.6. */
/*   (2 / N) sum_r <s_r gamma5 X gamma5 D_W s_r> = Tr(M_u^-1 X) + Tr(M_d^-1 X) */
/* from M_u + M_d = 2 D_W, "D_W the Dirac-Wilson operator without a twisted   */
/* mass term": in the kappa-normalised operator of O2 that is   */
/* D_W = M(mu = 0) = 1 - kappa D_hop.  Per source and timeslice, as written:  */
/*   L2_Gamma(t; s) = 2 sum_{x in t} sum_{alpha beta c}                       */
/*        conj(s_{alpha c}(x)) (gamma5 Gamma gamma5)_{alpha beta} (D_W s)_{beta c}(x). */
/* out is [16][Lt][2].                                                        */
/* ------------------------------------------------------------------------- */
void oracle_loops_gen_one_end(const int L[4], int theta, double kappa, const double *U, const double *s_, double *out_)
{
    const cplx *s = (const cplx *)s_;
    cplx *out = (cplx *)out_;
    const long V = vol(L), Vs = (long)L[0] * L[1] * L[2];
    const int T = L[3];
    cplx *y = malloc(V * SPINOR * sizeof(cplx));
    oracle_apply_M(L, theta, kappa, 0.0, U, s_, (double *)y);   /* D_W s */
    cplx g[5][4][4];
    build_gamma(g);
    for (int G = 0; G < 16; G++) {
        double gm[32];
        cplx Gam[4][4], t1[4][4], X5[4][4];
        oracle_gamma(G, gm);
        for (int i = 0; i < 4; i++)
            for (int j = 0; j < 4; j++) Gam[i][j] = gm[2 * (4 * i + j)] + I * gm[2 * (4 * i + j) + 1];
        mat4_mul(g[4], Gam, t1);
        mat4_mul(t1, g[4], X5);   /* gamma5 Gamma gamma5 */
        for (int t = 0; t < T; t++) {
            cplx acc = 0;
            for (long sx = 0; sx < Vs; sx++) {
                const long st = (long)t * Vs + sx;
                for (int al = 0; al < NS; al++)
                    for (int be = 0; be < NS; be++) {
                        if (X5[al][be] == 0) continue;
                        for (int c = 0; c < NC; c++)
                            acc += conj(s[(st * NS + al) * NC + c]) * X5[al][be] * y[(st * NS + be) * NC + c];
                    }
            }
            out[(long)G * T + t] = 2.0 * acc;
        }
    }
    free(y);
}

/* ------------------------------------------------------------------------- */
/* N3: Fourier transform of the loops ("the CUFFT  */
/* library" is used for it; the paper gives no formula).  Reading A25: for    */
/* integer triples n, spatial momentum p_i = 2 pi n_i / L_i, the plain        */
/* definition                                                                 */
/*   L_Gamma(t, p) = sum_{x in t} exp(+i p.x) sum_{alpha beta c}              */
/*        conj(eta_{alpha c}(x)) Gamma_{alpha beta} s_{beta c}(x)             */
/* (n = 0 is O6).  mom is [nmom][3], out is [nmom][16][Lt][2].                */
/* ------------------------------------------------------------------------- */
void oracle_loops_momentum(const int L[4], const double *eta_, const double *s_, int nmom, const int *mom, double *out_)
{
    const cplx *eta = (const cplx *)eta_, *s = (const cplx *)s_;
    cplx *out = (cplx *)out_;
    const long Vs = (long)L[0] * L[1] * L[2];
    const int T = L[3];
    const double twopi = 6.283185307179586476925286766559;
    for (int m = 0; m < nmom; m++)
        for (int G = 0; G < 16; G++) {
            double gm[32];
            oracle_gamma(G, gm);
            for (int t = 0; t < T; t++) {
                cplx acc = 0;
                for (long sx = 0; sx < Vs; sx++) {
                    const long st = (long)t * Vs + sx;
                    int x[4];
                    coords_of(L, st, x);
                    const double px = twopi * ((double)mom[3 * m] * x[0] / L[0] + (double)mom[3 * m + 1] * x[1] / L[1] +
                                               (double)mom[3 * m + 2] * x[2] / L[2]);
                    const cplx ph = cos(px) + I * sin(px);
                    cplx d = 0;
                    for (int a = 0; a < NS; a++)
                        for (int b = 0; b < NS; b++) {
                            const cplx gab = gm[2 * (4 * a + b)] + I * gm[2 * (4 * a + b) + 1];
                            if (gab == 0) continue;
                            for (int c = 0; c < NC; c++)
                                d += conj(eta[(st * NS + a) * NC + c]) * gab * s[(st * NS + b) * NC + c];
                        }
                    acc += ph * d;
                }
                out[((long)m * 16 + G) * T + t] = acc;
            }
        }
}
