// tsm_internal.cuh -- shared declarations of the CUDA path (sm_100a).
// Layouts, precision traits, load/store helpers, block reductions, context struct.
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/tsm.h"

// ------------------------------------------------------------------ geometry (H1)
// Division by a run-time lattice extent with a precomputed magic number (Granlund-Montgomery,
// exact for every 32-bit numerator): q = (t + ((n - t) >> 1)) >> (l - 1), t = umulhi(n, m).
struct FastDiv {
    unsigned m, l, d;
#ifdef __CUDACC__
    __device__ __forceinline__ unsigned div(unsigned n) const
    {
        if (l == 0) return n;
        const unsigned t = __umulhi(n, m);
        return (t + ((n - t) >> 1)) >> (l - 1);
    }
    __device__ __forceinline__ void divmod(unsigned n, unsigned& q, unsigned& r) const
    {
        q = div(n);
        r = n - q * d;
    }
#endif
};
inline FastDiv make_fastdiv(unsigned d)
{
    FastDiv f;
    f.d = d;
    unsigned l = 0;
    while ((1ull << l) < d) l++;
    f.l = l;
    f.m = l == 0 ? 0u : (unsigned)(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    return f;
}

struct Geom {
    int L[4];      // Lx, Ly, Lz, Lt (all even)
    int Lxh;       // Lx / 2
    int Vsh;       // Lx*Ly*Lz / 2: checkerboard sites per timeslice and parity
    int Vh;        // V / 2
    long long V;
    int theta;     // time boundary phase, +1 or -1 (A3)
    // stencil traversal order: z-slabs of bz planes, t sweeping inside a slab
    int bz;        // z planes per slab (divides Lz)
    int S;         // Lxh * Ly: cb sites per z plane
    FastDiv dLxh, dLy, dLz, dS, dSB, dLt;   // SB = bz * S
};

struct SiteCoord { int xh, y, z, t, rowpar; };

// cb index of parity `par` -> coordinates; x = 2*xh + rowpar, rowpar = (y+z+t+par)&1.
__device__ __forceinline__ SiteCoord decode_site(const Geom& g, int i, int par)
{
    SiteCoord s;
    unsigned r, xh, y, z, t;
    g.dLxh.divmod((unsigned)i, r, xh);
    g.dLy.divmod(r, r, y);
    g.dLz.divmod(r, t, z);
    s.xh = (int)xh; s.y = (int)y; s.z = (int)z; s.t = (int)t;
    s.rowpar = (s.y + s.z + s.t + par) & 1;
    return s;
}

// Traversal index v in [0, Vh) -> cb index i.  v runs over (z-slab, t, z in slab, y, xh): the sweep
// goes through all timeslices of one slab of bz z-planes before moving to the next slab, so the
// +-t neighbours of a site are only bz*S sites away in traversal order (the reuse window that has
// to stay in L2 is 2*bz*S sites instead of 2*Vsh).  Also returns the coordinates.
__device__ __forceinline__ int traverse_site(const Geom& g, int v, int par, SiteCoord& s)
{
    unsigned q1, r, zb, t, zi, rest, y, xh;
    g.dSB.divmod((unsigned)v, q1, r);
    g.dLt.divmod(q1, zb, t);
    g.dS.divmod(r, zi, rest);
    g.dLxh.divmod(rest, y, xh);
    s.xh = (int)xh; s.y = (int)y; s.z = (int)(zb * g.bz + zi); s.t = (int)t;
    s.rowpar = (s.y + s.z + s.t + par) & 1;
    return (int)(t * g.Vsh + s.z * g.S + rest);
}

__device__ __forceinline__ long long lex_of_site(const Geom& g, const SiteCoord& s)
{
    const int x = 2 * s.xh + s.rowpar;
    return x + (long long)g.L[0] * (s.y + (long long)g.L[1] * (s.z + (long long)g.L[2] * s.t));
}

// cb indices (in the other-parity field) of the 8 neighbours: nb[2*mu] = x+mu, nb[2*mu+1] = x-mu
__device__ __forceinline__ void neighbours(const Geom& g, int i, const SiteCoord& s, int nb[8])
{
    const int Lxh = g.Lxh, sy = g.Lxh, sz = g.Lxh * g.L[1], st = g.Vsh;
    nb[0] = s.rowpar ? (s.xh == Lxh - 1 ? i - (Lxh - 1) : i + 1) : i;
    nb[1] = s.rowpar ? i : (s.xh == 0 ? i + (Lxh - 1) : i - 1);
    nb[2] = (s.y == g.L[1] - 1) ? i - (g.L[1] - 1) * sy : i + sy;
    nb[3] = (s.y == 0) ? i + (g.L[1] - 1) * sy : i - sy;
    nb[4] = (s.z == g.L[2] - 1) ? i - (g.L[2] - 1) * sz : i + sz;
    nb[5] = (s.z == 0) ? i + (g.L[2] - 1) * sz : i - sz;
    nb[6] = (s.t == g.L[3] - 1) ? i - (g.L[3] - 1) * st : i + st;
    nb[7] = (s.t == 0) ? i + (g.L[3] - 1) * st : i - st;
}

// ------------------------------------------------------------------ precision traits
// A site's spinor is 24 reals r[2*q + ri], q = 3*alpha + c.  Storage: [chunk][cb] of 16-byte vectors.
template <int PREC> struct PT;
template <> struct PT<TSM_F64> {
    using real = double;
    static constexpr int NCHUNK = 12;   // double2 = one complex
    static constexpr int GAUGE_F64 = 1;
};
template <> struct PT<TSM_F32> {
    using real = float;
    static constexpr int NCHUNK = 6;    // float4 = two complex
    static constexpr int GAUGE_F64 = 0;
};
template <> struct PT<TSM_BF16> {
    using real = float;                 // arithmetic type
    static constexpr int NCHUNK = 3;    // 8 x bf16 = four complex
    static constexpr int GAUGE_F64 = 0;
};

// Storage is blocked: 32 consecutive cb sites form a block, inside a block the 16-byte vectors are
// ordered [chunk][site in block].  A warp still reads 512 contiguous bytes per chunk, a site's
// chunks sit at COMPILE-TIME offsets (k * 512 B) from one base address (one address computation per
// site instead of one per vector), and a block is one contiguous piece of memory.  Fields are
// padded to a whole number of blocks; kernels never touch the padding.
constexpr int FUSE_NTILES = 1024; // stencils on at most this many 128-site tiles finish their own norm reductions (section 6b)
constexpr int LB = 32;            // sites per layout block
constexpr int LB_ROW = LB * 16;   // bytes of one chunk row of a block
__host__ __device__ inline long long padded_sites(long long Vh) { return (Vh + LB - 1) / LB * LB; }
__host__ __device__ inline size_t field_bytes(int prec, long long Vh, int nrhs)
{
    const size_t per_site = prec == TSM_F64 ? 192 : (prec == TSM_F32 ? 96 : 48);
    return per_site * (size_t)padded_sites(Vh) * (size_t)nrhs;
}
// address of chunk 0 of site i in a field (or link pack) with NCH chunks per site
template <int NCH> __device__ __forceinline__ const char* site_ptr(const void* f, int i)
{
    return (const char*)f + (size_t)(i >> 5) * (size_t)(NCH * LB_ROW) + (size_t)((i & 31) * 16);
}
template <int NCH> __device__ __forceinline__ char* site_ptr(void* f, int i)
{
    return (char*)f + (size_t)(i >> 5) * (size_t)(NCH * LB_ROW) + (size_t)((i & 31) * 16);
}
__host__ __device__ inline int nchunk_of(int prec) { return prec == TSM_F64 ? 12 : (prec == TSM_F32 ? 6 : 3); }

__device__ __forceinline__ void bf16x8_to_float(const uint4& v, float* o)
{
    const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int j = 0; j < 4; j++) {
        o[2 * j] = __uint_as_float(w[j] << 16);
        o[2 * j + 1] = __uint_as_float(w[j] & 0xffff0000u);
    }
}
__device__ __forceinline__ uint4 float_to_bf16x8(const float* o)
{
    unsigned w[4];
#pragma unroll
    for (int j = 0; j < 4; j++) {
        __nv_bfloat162 b = __floats2bfloat162_rn(o[2 * j], o[2 * j + 1]);
        w[j] = *reinterpret_cast<unsigned*>(&b);
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}

// Load / store 8 consecutive reals (reals 8*k8 .. 8*k8+7 of site i) of a field.  NC: through the read-only
// path (ld.global.nc), valid only for data no thread writes during the kernel; NC = false is a plain coherent
// load (the CG residual that the RESID epilogue reads and then overwrites).
template <bool NC, typename V> __device__ __forceinline__ V ld16(const char* p)
{
    if constexpr (NC) return __ldg(reinterpret_cast<const V*>(p));
    else return *reinterpret_cast<const V*>(p);
}
template <int PREC, bool NC = true> __device__ __forceinline__ void load8(const void* f, int i, int k8, typename PT<PREC>::real* o)
{
    const char* p = site_ptr<PT<PREC>::NCHUNK>(f, i);
    if constexpr (PREC == TSM_F64) {
#pragma unroll
        for (int j = 0; j < 4; j++) { const double2 v = ld16<NC, double2>(p + (4 * k8 + j) * LB_ROW); o[2 * j] = v.x; o[2 * j + 1] = v.y; }
    } else if constexpr (PREC == TSM_F32) {
#pragma unroll
        for (int j = 0; j < 2; j++) { const float4 v = ld16<NC, float4>(p + (2 * k8 + j) * LB_ROW); o[4 * j] = v.x; o[4 * j + 1] = v.y; o[4 * j + 2] = v.z; o[4 * j + 3] = v.w; }
    } else {
        const uint4 v = ld16<NC, uint4>(p + k8 * LB_ROW);
        bf16x8_to_float(v, o);
    }
}
template <int PREC> __device__ __forceinline__ void store8(void* f, int i, int k8, const typename PT<PREC>::real* o)
{
    char* p = site_ptr<PT<PREC>::NCHUNK>(f, i);
    if constexpr (PREC == TSM_F64) {
#pragma unroll
        for (int j = 0; j < 4; j++) *reinterpret_cast<double2*>(p + (4 * k8 + j) * LB_ROW) = make_double2(o[2 * j], o[2 * j + 1]);
    } else if constexpr (PREC == TSM_F32) {
#pragma unroll
        for (int j = 0; j < 2; j++) *reinterpret_cast<float4*>(p + (2 * k8 + j) * LB_ROW) = make_float4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
    } else {
        *reinterpret_cast<uint4*>(p + k8 * LB_ROW) = float_to_bf16x8(o);
    }
}
template <int PREC, bool NC = true> __device__ __forceinline__ void load_spinor(const void* f, int i, typename PT<PREC>::real* s)
{
#pragma unroll
    for (int k = 0; k < 3; k++) load8<PREC, NC>(f, i, k, s + 8 * k);
}
template <int PREC> __device__ __forceinline__ void store_spinor(void* f, int i, const typename PT<PREC>::real* s)
{
#pragma unroll
    for (int k = 0; k < 3; k++) store8<PREC>(f, i, k, s + 8 * k);
}

// ------------------------------------------------------------------ gauge packs (H2)
// For output parity p and cb site i the pack holds 8 matrices, d = 2*mu + b:
//   b = 0: U_mu(x)          (forward hop)      b = 1: U_mu(x - mu)^dagger (backward hop, stored daggered)
// Same blocked storage as the fields ([block of 32 sites][chunk][site in block] of 16-byte vectors):
// fp64: 72 chunks of double2, link d = chunks 9d .. 9d+8 (row-major complex entries).
// fp32, 18 reals: 36 chunks of float4, direction mu = chunks 9mu .. 9mu+8 = 36 floats (fwd 18, bwd 18).
// fp32, 12 reals: 24 chunks of float4, link d = chunks 3d .. 3d+2 (rows 0,1; row 2 = conj(row0 x row1)).
__host__ __device__ inline int gauge_nchunk(int f64, int recon) { return f64 ? 72 : (recon == 18 ? 36 : 24); }
__host__ __device__ inline size_t gauge_pack_bytes(int f64, int recon, long long Vh)
{
    return (size_t)padded_sites(Vh) * 16 * gauge_nchunk(f64, recon);
}

template <typename T> __device__ __forceinline__ void reconstruct_row2(T* u)
{
    // u[0..11] rows 0,1 as (re,im) pairs; row2 = conj(row0 x row1)
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const T re = (u[2 * a] * u[6 + 2 * b] - u[2 * a + 1] * u[6 + 2 * b + 1]) - (u[2 * b] * u[6 + 2 * a] - u[2 * b + 1] * u[6 + 2 * a + 1]);
        const T im = (u[2 * a] * u[6 + 2 * b + 1] + u[2 * a + 1] * u[6 + 2 * b]) - (u[2 * b] * u[6 + 2 * a + 1] + u[2 * b + 1] * u[6 + 2 * a]);
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = -im;
    }
}

// Loads both links of direction mu for site i: uf = U_mu(x), ub = U_mu(x-mu)^dagger (18 reals each).
template <int PREC, int RECON> __device__ __forceinline__ void load_link_pair(const void* pack, int i, int mu,
                                                                             typename PT<PREC>::real* uf, typename PT<PREC>::real* ub)
{
    if constexpr (PT<PREC>::GAUGE_F64) {
        const char* p = site_ptr<72>(pack, i) + (18 * mu) * LB_ROW;
#pragma unroll
        for (int j = 0; j < 9; j++) { const double2 v = __ldcs(reinterpret_cast<const double2*>(p + j * LB_ROW)); uf[2 * j] = v.x; uf[2 * j + 1] = v.y; }
#pragma unroll
        for (int j = 0; j < 9; j++) { const double2 v = __ldcs(reinterpret_cast<const double2*>(p + (9 + j) * LB_ROW)); ub[2 * j] = v.x; ub[2 * j + 1] = v.y; }
    } else if constexpr (RECON == 18) {
        const char* p = site_ptr<36>(pack, i) + (9 * mu) * LB_ROW;
        float l[36];
#pragma unroll
        for (int j = 0; j < 9; j++) { const float4 v = __ldcs(reinterpret_cast<const float4*>(p + j * LB_ROW)); l[4 * j] = v.x; l[4 * j + 1] = v.y; l[4 * j + 2] = v.z; l[4 * j + 3] = v.w; }
#pragma unroll
        for (int j = 0; j < 18; j++) { uf[j] = l[j]; ub[j] = l[18 + j]; }
    } else {
        const char* p = site_ptr<24>(pack, i) + (6 * mu) * LB_ROW;
#pragma unroll
        for (int j = 0; j < 3; j++) { const float4 v = __ldcs(reinterpret_cast<const float4*>(p + j * LB_ROW)); uf[4 * j] = v.x; uf[4 * j + 1] = v.y; uf[4 * j + 2] = v.z; uf[4 * j + 3] = v.w; }
#pragma unroll
        for (int j = 0; j < 3; j++) { const float4 v = __ldcs(reinterpret_cast<const float4*>(p + (3 + j) * LB_ROW)); ub[4 * j] = v.x; ub[4 * j + 1] = v.y; ub[4 * j + 2] = v.z; ub[4 * j + 3] = v.w; }
        reconstruct_row2(uf);
        reconstruct_row2(ub);
    }
}

__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }

// o[c] = sum_c' U[c][c'] h[c'] for one spin row (3 complex), U 18 reals row-major; explicit FMA
// chains (12 per complex output: the compiler does not contract "x += a*b - c*d" into two FMAs).
template <typename T> __device__ __forceinline__ void su3_mul(const T* u, const T* h, T* o)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        T re = u[6 * c] * h[0];
        T im = u[6 * c] * h[1];
        re = fma_(-u[6 * c + 1], h[1], re);
        im = fma_(u[6 * c + 1], h[0], im);
        re = fma_(u[6 * c + 2], h[2], re);
        im = fma_(u[6 * c + 2], h[3], im);
        re = fma_(-u[6 * c + 3], h[3], re);
        im = fma_(u[6 * c + 3], h[2], im);
        re = fma_(u[6 * c + 4], h[4], re);
        im = fma_(u[6 * c + 4], h[5], im);
        re = fma_(-u[6 * c + 5], h[5], re);
        im = fma_(u[6 * c + 5], h[4], im);
        o[2 * c] = re;
        o[2 * c + 1] = im;
    }
}

// ------------------------------------------------------------------ Philox4x32-10 (H3, O3)
__device__ __forceinline__ uint32_t philox_word0(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return c0;
}
// 24 noise bits of site `lex` for source `sid`: component q uses bits 2q, 2q+1.
__device__ __forceinline__ uint32_t noise_bits(long long lex, uint64_t seed, uint32_t sid, int kind)
{
    return philox_word0((uint32_t)((uint64_t)lex & 0xffffffffu), (uint32_t)((uint64_t)lex >> 32), sid,
                        0x5A340000u | (uint32_t)kind, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32));
}
// eta component as (re, im) from its 2-bit code: Z4 -> i^k, Z2 -> 1 - 2(k&1).
__device__ __forceinline__ void noise_value(int k, int kind, float& re, float& im)
{
    if (kind == TSM_Z4) {
        re = (k == 0) ? 1.f : (k == 2 ? -1.f : 0.f);
        im = (k == 1) ? 1.f : (k == 3 ? -1.f : 0.f);
    } else {
        re = (k & 1) ? -1.f : 1.f;
        im = 0.f;
    }
}

// ------------------------------------------------------------------ block reduction (A19)
// Deterministic: fixed shuffle tree inside a warp, then a fixed serial sum over warps.
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
// Sum over the threads of one threadIdx.y row (blockDim.x a multiple of 32, <= 1024).
// Result valid in threadIdx.x == 0.  smem: at least 32 * blockDim.y doubles.
__device__ __forceinline__ double block_row_sum(double v, double* smem)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    v = warp_sum(v);
    double* row = smem + 32 * threadIdx.y;
    if (lane == 0) row[w] = v;
    __syncthreads();
    double t = 0;
    if (threadIdx.x == 0)
        for (int k = 0; k < nw; k++) t += row[k];
    __syncthreads();
    return t;
}

// Per-source CG scalars, device resident (A14: every source has its own).
struct CgScalars {
    double rr[TSM_MAX_NRHS];      // |r|^2 of the current residual
    double bb[TSM_MAX_NRHS];      // |b'|^2
    double pq[TSM_MAX_NRHS];      // Re <p, q>
    double beta[TSM_MAX_NRHS];
    double alpha[TSM_MAX_NRHS];   // rr / Re<p,q> of this iteration; 0 for a frozen source
    double rr_new[TSM_MAX_NRHS];  // |r|^2 after this iteration's residual update
    // N4 mixed-precision solver: state of the fp64 defect-correction loop around the fp32 CG
    double bb_outer[TSM_MAX_NRHS], rr_outer[TSM_MAX_NRHS];
    int iters_outer[TSM_MAX_NRHS];
    int outer_done[TSM_MAX_NRHS];   // 0 live, 1 converged, 2 broken down
    int all_outer_done;
    int iters[TSM_MAX_NRHS];
    int done[TSM_MAX_NRHS];       // frozen: converged, broken down, or zero source
    int status[TSM_MAX_NRHS];
    int all_done;
    int sticky_breakdown;         // set by any breakdown, cleared only by tsm_run_loop_set (its LP batches are not waited for one by one)
    int loop_left;                // iterations the device-side loop (WHILE node of the CG graph) may still run
    unsigned ticket;              // last-block counter, always left at 0
};

// ------------------------------------------------------------------ epilogue coefficients
// out = Tx * x + Td * (D in), T = c_up on spins 0,1 and c_lo on spins 2,3 (complex), i.e.
// T = alpha + i beta gamma5 with c_up = alpha + i beta, c_lo = alpha - i beta (C3: gamma5 diagonal).
// stencil epilogues beyond out = Tx x + Td D in
enum { EPI_NONE = 0, EPI_NORM = 1, EPI_RESID = 2 };
struct TwistCoef { double up_re, up_im, lo_re, lo_im; };
struct DslashCoef { TwistCoef x, d; };

// o = c (x) v on reals 8 k8 .. 8 k8 + 7 of a site (c.up on spins 0, 1, c.lo on spins 2, 3): the arithmetic of k_twist,
// shared with the whole-solve persistent kernel (dslash_small.cu) so that both give the same bits
template <typename T> __device__ __forceinline__ void twist8(const TwistCoef& c, const int k8, const T* v, T* o)
{
#pragma unroll
    for (int j = 0; j < 4; j++) {
        const int q = 4 * k8 + j;
        const T cr = (T)(q < 6 ? c.up_re : c.lo_re), ci = (T)(q < 6 ? c.up_im : c.lo_im);
        // explicit FMAs: left to the compiler, "a b - c d" is contracted differently in different kernels
        o[2 * j] = fma_(-ci, v[2 * j + 1], cr * v[2 * j]);
        o[2 * j + 1] = fma_(ci, v[2 * j], cr * v[2 * j + 1]);
    }
}

// ------------------------------------------------------------------ context
struct GammaTable {          // Gamma_{alpha, col[alpha]} = i^ph[alpha], all other entries 0
    int col[16][4];
    int ph[16][4];
};

// Optional per-launch timing (tsm_profile): CUDA events on the library's stream around each
// stencil / BLAS launch.  kind: 0 stencil, 1 stencil+xpay, 2 stencil+xpay+norm, 3 stencil+xpay+residual update, 4 update_xp.
struct ProfRec { int prec, kind, nrhs; cudaEvent_t a, b; };

// A captured run of CG iterations (CUDA graph), keyed by everything the captured launches depend on.  iters > 0: that
// many iterations in a row; iters == 0: ONE iteration as the body of a WHILE node, repeated on the device until
// every source is frozen or cg->loop_left runs out (no host round trip for the stopping test).
struct CgGraph {
    int prec, nrhs, iters;
    void *x, *r, *p, *w, *t;
    double tol;
    long long launches;              // kernels inside the graph
    cudaGraphExec_t exec;
};

// Tensor maps (4 x 128 B, opaque here) of a field the box stencil has read before, keyed by its address.
struct BoxMapCache {
    const void* field;
    int nrhs;
    alignas(64) char maps[4 * 128];
};

struct tsm_ctx {
    Geom g;
    int device;
    cudaStream_t stream;             // where work is enqueued: the caller's stream or own_stream
    cudaStream_t own_stream;         // library-owned BLOCKING stream (serialises with the legacy default stream)
    std::vector<CgGraph> graphs;     // cleared whenever kappa/mu, the gauge storage or the workspace change
    std::vector<BoxMapCache> box_maps;
    int stencil_choice;              // tsm_set_stencil_kernel: 0 automatic, 1 k_dslash, 2 k_dslash_tile, 3 k_dslash_box, 5 k_dslash_small
    int graphs_on;                   // tsm_set_graphs: 0 off, 1 chunks of 4 iterations, 2 device-side loop, 3 persistent kernel, 4 automatic
    long long loop_per_pass;         // launch accounting of the last device-side loop: kernels per pass (0: none pending),
    int loop_eager, loop_nrhs;       // iterations run before the loop, sources of that solve (settled when the scalars are read)
    // per solution slot: what tsm_solve_wait needs to report on a solve that was only enqueued (tsm_solve_async)
    CgScalars* cg_snap[2];           // pinned copies of the CG scalars, made on the stream right after the solve
    cudaEvent_t slot_ev0[2], slot_ev1[2];
    double slot_tol[2];
    bool slot_pending[2];
    long long slot_loop_per_pass[2];
    int slot_loop_eager[2];
    double kappa, mu;
    bool have_params, have_gauge, have_ws;
    int recon;                       // storage of the fp32 link copy (18 / 12)
    int max_nrhs;
    int ws_prec;                     // TSM_F64: full workspace; TSM_F32: low-precision-only (no fp64 packs, fp32-sized vectors)
    int nsm;
    // workspace carving (device pointers into the caller's buffer)
    char* ws;
    size_t ws_bytes;
    void* gauge64[2];                // fp64 packs for output parity 0 / 1
    void* gauge32[2];                // fp32 packs
    void* staging;                   // raw host-layout staging (links or spinors), fp64
    size_t staging_bytes;
    void* vec[6];                    // solver vectors r, p, b (mixed solver only), w, t, aux: single-parity, max_nrhs, fp64-sized
    void* slot[2];                   // solutions: [parity][rhs][chunk][cb], fp64-sized
    int slot_prec[2], slot_nrhs[2], slot_kind[2];
    uint64_t slot_seed[2];
    uint32_t slot_ids[2][TSM_MAX_NRHS];
    double* partials;                // reduction scratch of the BLAS / contraction kernels
    size_t partials_count;
    double* norm_partials;           // [rhs][tile] sums of |out|^2 left by the stencil's NORM epilogue
    size_t norm_partials_count;
    int norm_ntiles;
    bool norm_reduced;               // the last stencil launch finished its own reduction (k_dslash_small): skip k_cg_reduce
    double* loops_src[2];            // per-source loops of a slot [rhs][n_ops][T][2]
    double* acc_corr;                // [n_ops][T][2]
    double* acc_lp;
    double* loops_out;               // finalize output
    // library-owned small allocations
    CgScalars* cg;                   // device
    CgScalars* cg_host;              // pinned
    double* host_small;              // pinned scratch (loops, unitarity)
    uint32_t* ids_dev;               // [2][TSM_MAX_NRHS]
    GammaTable gam;
    int n_ops, with_deriv, with_one_end, with_gen_one_end, with_momenta, n_hp, n_lp;
    bool loops_ready;                // the Eq. 2.4 accumulators are zeroed / consistent with n_ops (tsm_loops_reset)
    int hp_prec;                     // TSM_F64 or TSM_MIXED (tsm_set_hp_precision)
    int n_mom, mom[TSM_MAX_MOMENTA][3];   // momenta of the projected loops (tsm_loops_set_momenta)
    long long launches;
    bool prof_on;
    std::vector<ProfRec> prof;
    std::vector<cudaEvent_t> prof_pool;
    cudaEvent_t ev0, ev1;
    std::string err;
};

#define TSM_CUDA(ctx, expr)                                                                      \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                     \
            return TSM_ECUDA;                                                                    \
        }                                                                                        \
    } while (0)

inline int prof_begin(tsm_ctx* ctx, int prec, int kind, int nrhs)
{
    if (!ctx->prof_on) return -1;
    ProfRec r{prec, kind, nrhs, nullptr, nullptr};
    for (cudaEvent_t* e : {&r.a, &r.b}) {
        if (!ctx->prof_pool.empty()) { *e = ctx->prof_pool.back(); ctx->prof_pool.pop_back(); }
        else if (cudaEventCreate(e) != cudaSuccess) return -1;
    }
    cudaEventRecord(r.a, ctx->stream);
    ctx->prof.push_back(r);
    return (int)ctx->prof.size() - 1;
}
inline void prof_end(tsm_ctx* ctx, int idx)
{
    if (idx >= 0) cudaEventRecord(ctx->prof[idx].b, ctx->stream);
}

inline int tsm_fail(tsm_ctx* ctx, int code, const char* msg)
{
    if (ctx) ctx->err = msg;
    return code;
}

// ------------------------------------------------------------------ launchers (defined in the .cu files)
int launch_dslash(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x,
                  void* out, const DslashCoef& c, int mode);
int launch_dslash_tile(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x,
                       void* out, const DslashCoef& c, int mode);
int launch_dslash_small(tsm_ctx* ctx, int prec, int out_parity, bool dagger, int nrhs, const void* in, const void* x,
                        void* out, const DslashCoef& c, int mode);
int launch_dslash_box(tsm_ctx* ctx, int out_parity, bool dagger, int nrhs, const void* in, const void* x, void* out,
                      const DslashCoef& c, int mode);
bool box_stencil_supported(const tsm_ctx* ctx);
int launch_twist(tsm_ctx* ctx, int prec, int nrhs, const void* in, void* out, const TwistCoef& c);
int launch_gauge_pack(tsm_ctx* ctx, double* max_dev_out);
int launch_pack_spinor(tsm_ctx* ctx, int prec, int nrhs, const double* dev_lex, void* dev_native, size_t par_stride = 0);
int launch_unpack_spinor(tsm_ctx* ctx, int prec, int nrhs, const void* dev_native, double* dev_lex, size_t par_stride = 0);
int launch_noise(tsm_ctx* ctx, int prec, int nrhs, uint64_t seed, const uint32_t* dev_ids, int kind, void* dev_full);
int launch_cg_init(tsm_ctx* ctx, int prec, int nrhs, const void* r, void* p, void* x);
int launch_cg_reduce(tsm_ctx* ctx, int which, int nrhs, int force = 0);
int launch_mixed_ctl(tsm_ctx* ctx, int mode, int nrhs, double tol);
int launch_mixed_axpy(tsm_ctx* ctx, int nrhs, void* x64, const void* e32);
int launch_cg_update_xp(tsm_ctx* ctx, int prec, int nrhs, void* x, void* p, const void* r, double tol, unsigned long long loop = 0,
                        int in_loop = 0);
int launch_cg_loop_begin(tsm_ctx* ctx, int n);
// arguments of the persistent CG kernels (dslash.cu: 128-site tiles, k_dslash's arithmetic; dslash_small.cu: 32-site
// blocks, k_dslash_small's arithmetic)
struct PcgArgs {
    Geom g;
    int nrhs, ntiles, slab, max_iter;   // ntiles: 128-site tiles, or 32-site blocks for the small form
    double tol;
    const void* pack[2];            // link packs of output parity 0 / 1
    void *x, *r, *p, *w, *t;
    DslashCoef c1, c2, c3, c4;      // the four stencil launches of cg_iteration (api_solve.cu)
    double* partials;               // [2][nrhs][ntiles]: |w|^2 per tile, |r|^2 per tile
    CgScalars* cg;
    // whole-solve form (small kernel only): source preparation, CG initialisation and reconstruction in the same launch
    int whole;                      // 0: the iteration loop only
    void *s_o, *aux;                // the slot's odd half (eta_o on entry, s_o on exit); scratch vector
    TwistCoef tw_rinv;              // aux = R^-1 eta_o
    DslashCoef cp1, cp2, cp3, crec; // bhat, t, b' (tsm_solve's three preparation stencils) and the reconstruction
    double* init_groups;            // [nrhs][3 ntiles]: |r|^2 of every (32-site block, group of 8 reals)
    int init_gx;                    // blocks of k_cg_init's grid on this lattice (its summation order is reproduced)
};
int launch_cg_persistent_small(tsm_ctx* ctx, int prec, PcgArgs& a);
bool cg_persistent_supported(const tsm_ctx* ctx, int prec, int nrhs);
bool cg_persistent_preferred(const tsm_ctx* ctx, int prec, int nrhs);
int launch_cg_persistent(tsm_ctx* ctx, int prec, int nrhs, void* x, void* r, void* p, void* w, void* t, const DslashCoef& c1,
                         const DslashCoef& c2, const DslashCoef& c3, const DslashCoef& c4, double tol, int max_iter,
                         const PcgArgs* whole = nullptr);
int blas_grid_x(const tsm_ctx* ctx);
int launch_convert(tsm_ctx* ctx, int prec_in, int prec_out, int nrhs_fields, const void* in, void* out);
int launch_contract(tsm_ctx* ctx, int slot);
int launch_accumulate(tsm_ctx* ctx, double* acc, const double* a, const double* b, int nrhs);
int launch_finalize(tsm_ctx* ctx);
void build_gamma_table(GammaTable& t);
int ctx_enter(tsm_ctx* ctx, bool need_ws, bool need_gauge, bool need_params);
void ctx_drop_graphs(tsm_ctx* ctx);
// |a - b|^2 per source over full-lattice fp64 fields, left in cg->pq[rhs] (true-residual helper)
int launch_diff_norm2(tsm_ctx* ctx, int nrhs, const void* a, const void* b);
