// dslash_box.cu -- H5 for fp32 batches: the stencil with the neighbour spinors of a 4-D tile staged in shared
// memory by tensor-map TMA boxes and the links of the tile held in registers.
//
// Why: with the links amortised over 12 sources the batched stencil of dslash_tile.cu is
// bound by the SM <- L2 fabric, not by HBM: its 1-D tiles (8 y rows of one (z,t)) pull ~5.75 input sites per output
// site through L2 and run at the ~6300 B/clk the fabric delivers chip-wide.  Here a tile is 4-D,
//
//     (all x of rpb = 32 / Lxh rows of y)  x  2 planes of z  x  2 planes of t   =  128 output sites = 4 layout blocks,
//
// so the other-parity sites it needs are its own 4 blocks plus one halo row / block on each y, z, t face: 4.0 input
// sites per output site, each crossing L2 -> SM once per tile and source.  In the blocked field layout
// [block of 32 cb sites][chunk][site] such a tile and each of its halos IS a 5-D box (128 floats, chunk, y block, z,
// t x rhs) of the field, periodic wrap being nothing but the box's start coordinate: seven cp.async.bulk.tensor
// loads per (tile, source) fill one 48 KB stage of a 4-stage ring; the stage of iteration i + 4 is issued by the
// lane that is LAST to finish reading stage i (a shared-memory ticket), so nobody ever waits for a free stage.
//
// Arithmetic: 256 threads = 4 blocks x 2 direction pairs x 32 sites.  Warp (b, P) keeps the four links
// U_mu(x), U_mu(x-mu)^dag, mu = 2P, 2P+1, of its 32 sites in REGISTERS for the whole tile (72 floats; loaded once per
// tile, 12-real links rebuilt once per tile), so the per-source inner loop reads only spinors from shared memory
// (LDS.128, conflict free) -- the 576 B of link reads per site and source that kept the LSU of dslash_tile.cu at 76 %
// are gone.  The two warps of a block pair exchange half of their 24 partial sums through shared memory (warp P
// keeps spins 2P, 2P+1), one 64-thread named barrier per source, and each finishes 12 reals of the site: twist / x
// term / norm / residual epilogues as in dslash.cu, on whole 16-byte chunks 3P .. 3P+2.
//
// A source's result is a fixed sequence of operations whatever batch it is in (A14): the library routes EVERY fp32
// stencil of a context with max_nrhs >= 2 here when the lattice fits (32 % Lxh == 0, Ly % rpb == 0), single sources
// included.  Sums across sites stay fp64 with fixed trees (A19): each warp leaves one partial per (source, tile).
#include <cuda.h>
#include <cstdlib>
#include <cstring>

#include "bulk_copy.cuh"
#include "dslash_common.cuh"

namespace {

constexpr int BT = 128;        // sites per tile
constexpr int BTHREADS = 256;  // 4 blocks x 2 direction pairs x 32 sites
constexpr int NST_MAX = 4;     // stages of the spinor ring (3 when a stage is 60 KB: Lxh = 32)
constexpr int NCH32 = 6;       // float4 chunks of an fp32 spinor
constexpr int CB = NCH32 * LB_ROW;   // bytes of one layout block of an fp32 field (3072)
constexpr int BOX_R = 1;       // sources per pass of a warp (2 was measured slower: 944 vs 859 us)
constexpr size_t XBUF_BYTES = 4 * 2 * BOX_R * 3 * LB_ROW;   // exchange buffers: [block][half][source of the pass][3 chunks][32 sites]
constexpr size_t SMEM_MAX = 224 * 1024;

struct BoxGeom {
    int lxs;          // log2(Lxh)
    int Lxh, rpb, nyb, Lz, Lt, Lzh, Lth;
    int HB;           // bytes of one halo row in a stage: NCH * Lxh * 16
    int stage_bytes;  // 12 CB + 8 HB
    int nst;          // stages of the ring that fit beside the exchange buffers
    int ntiles;       // nyb * Lzh * Lth
    int Zs;           // tiles (z pairs) per z slab of the traversal
    FastDiv d_nyb, d_Zs, d_Lth;
};

struct BoxMaps { CUtensorMap center, yrow, zface, tface; };

__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, int c4, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(
                     smem_u32(dst)),
                 "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
                 : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// stage layout (bytes): centre blocks [tt][zz] at (2 tt + zz) CB; then the z-, z+, t-, t+ halo blocks, then the
// y-, y+ halo rows [tt][zz] of HB bytes each
__device__ __forceinline__ int off_zm(int tt) { return (4 + tt) * CB; }
__device__ __forceinline__ int off_zp(int tt) { return (6 + tt) * CB; }
__device__ __forceinline__ int off_tm(int zz) { return (8 + zz) * CB; }
__device__ __forceinline__ int off_tp(int zz) { return (10 + zz) * CB; }

// Traversal: tile index -> (y block fastest, z pair inside a slab of Zs pairs, t pair, z slab).  The chip's CTAs
// work on consecutive tiles, i.e. on a front of a few t pairs of one z slab, so a tile's y and t halos, and its z halos
// inside the slab, are the centre blocks of tiles of the same or the previous wave (L2 hits); only the z faces of a
// slab are fetched from DRAM twice.
struct TileCoord { int yb, z0, t0; };
__device__ __forceinline__ TileCoord tile_coord(const BoxGeom& bg, int tile)
{
    unsigned q, yb, zi, tp, zs;
    bg.d_nyb.divmod((unsigned)tile, q, yb);
    bg.d_Zs.divmod(q, q, zi);
    bg.d_Lth.divmod(q, zs, tp);
    return {(int)yb, 2 * (int)(zs * bg.Zs + zi), 2 * (int)tp};
}

// the seven boxes of (tile, first source rhs0 + src) into stage `st`, signalled on `bar`
__device__ __forceinline__ void issue_stage(const BoxGeom& bg, const BoxMaps& m, char* st, uint64_t* bar, int tile, int src)
{
    const TileCoord tc = tile_coord(bg, tile);
    const int tb = src * bg.Lt;   // dimension 4 of the maps is t + Lt * rhs
    const int zm = tc.z0 == 0 ? bg.Lz - 1 : tc.z0 - 1, zp = tc.z0 + 2 == bg.Lz ? 0 : tc.z0 + 2;
    const int tm = tc.t0 == 0 ? bg.Lt - 1 : tc.t0 - 1, tp = tc.t0 + 2 == bg.Lt ? 0 : tc.t0 + 2;
    const int ybm = tc.yb == 0 ? bg.nyb - 1 : tc.yb - 1, ybp = tc.yb + 1 == bg.nyb ? 0 : tc.yb + 1;
    mbar_expect_tx(bar, (unsigned)bg.stage_bytes);
    tma_load_5d(st, &m.center, 0, 0, tc.yb, tc.z0, tb + tc.t0, bar);
    tma_load_5d(st + off_zm(0), &m.zface, 0, 0, tc.yb, zm, tb + tc.t0, bar);
    tma_load_5d(st + off_zp(0), &m.zface, 0, 0, tc.yb, zp, tb + tc.t0, bar);
    tma_load_5d(st + off_tm(0), &m.tface, 0, 0, tc.yb, tc.z0, tb + tm, bar);
    tma_load_5d(st + off_tp(0), &m.tface, 0, 0, tc.yb, tc.z0, tb + tp, bar);
    tma_load_5d(st + 12 * CB, &m.yrow, (bg.rpb - 1) * bg.Lxh * 4, 0, ybm, tc.z0, tb + tc.t0, bar);
    tma_load_5d(st + 12 * CB + 4 * bg.HB, &m.yrow, 0, 0, ybp, tc.z0, tb + tc.t0, bar);
}

__device__ __forceinline__ void lds_spinor(const char* p, int cs, float* psi)
{
#pragma unroll
    for (int k = 0; k < 6; k++) {
        const float4 v = *reinterpret_cast<const float4*>(p + k * cs);
        psi[4 * k] = v.x; psi[4 * k + 1] = v.y; psi[4 * k + 2] = v.z; psi[4 * k + 3] = v.w;
    }
}

// the two links of direction mu of site (block gb, lane j) from the fp32 pack into uf / ub (18 reals each)
template <int RECON> __device__ __forceinline__ void ldg_link_pair(const char* pack, size_t gb, int j, int mu, float* uf, float* ub)
{
    constexpr int NCHG = RECON == 18 ? 36 : 24;
    const char* p = pack + gb * (size_t)(NCHG * LB_ROW) + j * 16;
    if constexpr (RECON == 18) {
        float l[36];
#pragma unroll
        for (int k = 0; k < 9; k++) {
            const float4 v = __ldcs(reinterpret_cast<const float4*>(p + (9 * mu + k) * LB_ROW));
            l[4 * k] = v.x; l[4 * k + 1] = v.y; l[4 * k + 2] = v.z; l[4 * k + 3] = v.w;
        }
#pragma unroll
        for (int k = 0; k < 18; k++) { uf[k] = l[k]; ub[k] = l[18 + k]; }
    } else {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const float4 v = __ldcs(reinterpret_cast<const float4*>(p + (6 * mu + k) * LB_ROW));
            uf[4 * k] = v.x; uf[4 * k + 1] = v.y; uf[4 * k + 2] = v.z; uf[4 * k + 3] = v.w;
        }
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const float4 v = __ldcs(reinterpret_cast<const float4*>(p + (6 * mu + 3 + k) * LB_ROW));
            ub[4 * k] = v.x; ub[4 * k + 1] = v.y; ub[4 * k + 2] = v.z; ub[4 * k + 3] = v.w;
        }
    }
}

struct BoxArgs {
    BoxGeom bg;
    int par, nrhs, theta, check_done;
    const char* pack;
    const char* x;
    char* out;
    DslashCoef cf;
    double* partials;
    const CgScalars* cg;
};

// one hop for up to R sources: all neighbour spinors are requested first, then the arithmetic (the link is shared)
template <int MU, int SGN, int R>
__device__ __forceinline__ void hop_r(const char* const* st, int nact, int off, int cs, const float* u, float ph, float (*acc)[24])
{
#pragma unroll
    for (int r = 0; r < R; r++)
        if (r < nact) {
            float psi[24], h[12], gq[12];
            lds_spinor(st[r] + off, cs, psi);
            project<float, MU, SGN>(psi, h);
            if (MU == 3 && ph != 1.f) rscale_f32<6>(ph, h);   // time-boundary phase (A22); skipping a multiplication by one is exact
            su3_mul(u, h, gq);
            su3_mul(u, h + 6, gq + 6);
            accumulate<float, MU, SGN>(gq, acc[r]);
        }
}

// The work of one warp: P = 0 hops in x and y, P = 1 hops in z and t; keeps spins 2P, 2P+1 of the result.
// Every pass of the loop handles up to R consecutive sources of the tile (two independent instruction streams per
// warp: with 8 warps per SM the second stream is what hides the shared-memory and FMA latencies).
template <int RECON, bool DAGGER, bool XPAY, int EPI, int P, int R>
__device__ __forceinline__ void run_warp(const BoxArgs& a, const BoxMaps& maps, char* smem, uint64_t* full, unsigned* ticket, char* xbuf)
{
    constexpr int SF = DAGGER ? +1 : -1;   // forward hop carries (1 - g_mu), dagger swaps
    const BoxGeom& bg = a.bg;
    const int j = threadIdx.x & 31, w = threadIdx.x >> 5, b = w >> 1;
    const int tt = b >> 1, zz = b & 1;
    const int ry = j >> bg.lxs, xh = j & (bg.Lxh - 1);
    const size_t fb = (size_t)bg.ntiles * 4 * CB;   // bytes of one source of an fp32 single-parity field (V_h = 32 * blocks)
    const float cdr = (float)(P == 0 ? a.cf.d.up_re : a.cf.d.lo_re), cdi = (float)(P == 0 ? a.cf.d.up_im : a.cf.d.lo_im);
    const float cxr = (float)(P == 0 ? a.cf.x.up_re : a.cf.x.lo_re), cxi = (float)(P == 0 ? a.cf.x.up_im : a.cf.x.lo_im);
    const bool d_real = cdi == 0.f;
    const int my_tiles = ((int)blockIdx.x < bg.ntiles) ? (bg.ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const int n_iter = my_tiles * a.nrhs;   // (tile, source) pairs of this CTA, in order

    float u[4][18];
    int off[4], cs[4];
    float ph_f = 1.f, ph_b = 1.f;
    size_t gb = 0;
    int tile = blockIdx.x, src = 0;
    int stage = 0;
    unsigned phase = 0;
    const int NST = bg.nst;

    auto load_links = [&](int which, size_t gblk) {   // which = 0: direction 2P, 1: direction 2P + 1
        ldg_link_pair<RECON>(a.pack, gblk, j, 2 * P + which, u[2 * which], u[2 * which + 1]);
    };
    auto block_of = [&](int tl) -> size_t {
        const TileCoord tc = tile_coord(bg, tl);
        return ((size_t)(tc.t0 + tt) * bg.Lz + (tc.z0 + zz)) * bg.nyb + tc.yb;
    };

    for (int it = 0; it < n_iter;) {
        if (src == 0) {
            const TileCoord tc = tile_coord(bg, tile);
            gb = ((size_t)(tc.t0 + tt) * bg.Lz + (tc.z0 + zz)) * bg.nyb + tc.yb;
            if (it == 0) { load_links(0, gb); load_links(1, gb); }   // later tiles: loaded during the previous tile's last pass
            if (RECON == 12) {
#pragma unroll
                for (int k = 0; k < 4; k++) reconstruct_row2(u[k]);
            }
            const int y = tc.yb * bg.rpb + ry, t = tc.t0 + tt;
            const int rowpar = (y + tc.z0 + zz + t + a.par) & 1;
            if (P == 0) {
                const int xf = rowpar ? ((xh + 1) & (bg.Lxh - 1)) : xh, xb = rowpar ? xh : ((xh - 1) & (bg.Lxh - 1));
                off[0] = b * CB + ((ry << bg.lxs) + xf) * 16; cs[0] = LB_ROW;
                off[1] = b * CB + ((ry << bg.lxs) + xb) * 16; cs[1] = LB_ROW;
                if (ry + 1 < bg.rpb) { off[2] = b * CB + (j + bg.Lxh) * 16; cs[2] = LB_ROW; }
                else { off[2] = 12 * CB + (4 + b) * bg.HB + xh * 16; cs[2] = bg.Lxh * 16; }
                if (ry >= 1) { off[3] = b * CB + (j - bg.Lxh) * 16; cs[3] = LB_ROW; }
                else { off[3] = 12 * CB + b * bg.HB + xh * 16; cs[3] = bg.Lxh * 16; }
            } else {
                off[0] = (zz == 0 ? (2 * tt + 1) * CB : off_zp(tt)) + j * 16;
                off[1] = (zz == 1 ? (2 * tt) * CB : off_zm(tt)) + j * 16;
                off[2] = (tt == 0 ? (2 + zz) * CB : off_tp(zz)) + j * 16;
                off[3] = (tt == 1 ? zz * CB : off_tm(zz)) + j * 16;
                cs[0] = cs[1] = cs[2] = cs[3] = LB_ROW;
                ph_f = (t == bg.Lt - 1) ? (float)a.theta : 1.f;
                ph_b = (t == 0) ? (float)a.theta : 1.f;
            }
        }
        const int nact = a.nrhs - src < R ? a.nrhs - src : R;   // sources of this pass (warp-uniform)
        const bool last_pass = src + nact == a.nrhs;
        const bool more = last_pass && it + nact < n_iter;             // another tile follows: fetch its links early
        const size_t gb_next = more ? block_of(tile + gridDim.x) : 0;
        const size_t o_site = (size_t)src * fb + gb * CB + j * 16 + (3 * P) * LB_ROW;

        const char* st[R];
        int stg[R];
        {
            int s_ = stage;
            unsigned ph_ = phase;
#pragma unroll
            for (int r = 0; r < R; r++) {
                stg[r] = s_;
                st[r] = smem + (size_t)s_ * bg.stage_bytes;
                if (r < nact) mbar_wait(&full[s_], ph_);
                if (++s_ == NST) { s_ = 0; ph_ ^= 1u; }
                if (r + 1 == nact) { stage = s_; phase = ph_; }
            }
        }
        float acc[R][24];
#pragma unroll
        for (int r = 0; r < R; r++)
#pragma unroll
            for (int k = 0; k < 24; k++) acc[r][k] = 0.f;
        {
            hop_r<2 * P, SF, R>(st, nact, off[0], cs[0], u[0], 1.f, acc);
            hop_r<2 * P, -SF, R>(st, nact, off[1], cs[1], u[1], 1.f, acc);
            if (more) load_links(0, gb_next);
            hop_r<2 * P + 1, SF, R>(st, nact, off[2], cs[2], u[2], ph_f, acc);
            hop_r<2 * P + 1, -SF, R>(st, nact, off[3], cs[3], u[3], ph_b, acc);
            if (more) load_links(1, gb_next);
        }

        // the epilogue's own-site inputs: requested now, used after the exchange
        float xv[R][12], rv[R][12];
#pragma unroll
        for (int r = 0; r < R; r++) {
            if (XPAY && r < nact) {
#pragma unroll
                for (int k = 0; k < 3; k++) {
                    const float4 v = __ldg(reinterpret_cast<const float4*>(a.x + o_site + r * fb + k * LB_ROW));
                    xv[r][4 * k] = v.x; xv[r][4 * k + 1] = v.y; xv[r][4 * k + 2] = v.z; xv[r][4 * k + 3] = v.w;
                }
            }
            if (EPI == EPI_RESID && r < nact) {   // out is the CG residual r: coherent loads (it is rewritten below)
#pragma unroll
                for (int k = 0; k < 3; k++) {
                    const float4 v = *reinterpret_cast<const float4*>(a.out + o_site + r * fb + k * LB_ROW);
                    rv[r][4 * k] = v.x; rv[r][4 * k + 1] = v.y; rv[r][4 * k + 2] = v.z; rv[r][4 * k + 3] = v.w;
                }
            }
        }

        // this warp is done with the stages; the last of the 8 warps to say so refills a stage for ordinal + NST
        __syncwarp();
        if (j == 0) {
            __threadfence_block();
#pragma unroll
            for (int r = 0; r < R; r++) {
                if (r >= nact) break;
                const unsigned old = atomicAdd(&ticket[stg[r]], 1u);
                if ((old & 7u) == 7u) {
                    __threadfence_block();
                    const int it2 = it + r + NST;
                    if (it2 < n_iter) {
                        int src2 = src + r + NST, tile2 = tile;
                        while (src2 >= a.nrhs) { src2 -= a.nrhs; tile2 += gridDim.x; }
                        issue_stage(bg, maps, smem + (size_t)stg[r] * bg.stage_bytes, &full[stg[r]], tile2, src2);
                        if (src2 == 0) {   // first source of a tile: pull that tile's links into L2 ahead of the warps' loads
                            const TileCoord tc = tile_coord(bg, tile2);
                            constexpr unsigned LBYTES = (RECON == 18 ? 36 : 24) * LB_ROW;
#pragma unroll
                            for (int q = 0; q < 4; q++) {
                                const size_t g2 = ((size_t)(tc.t0 + (q >> 1)) * bg.Lz + (tc.z0 + (q & 1))) * bg.nyb + tc.yb;
                                prefetch_l2(a.pack + g2 * LBYTES, LBYTES);
                            }
                        }
                    }
                }
            }
        }

        // exchange: warp P keeps reals 12P .. 12P+11 (spins 2P, 2P+1) of every source and hands the other 12 to its
        // partner.  One buffer per block pair: the first barrier says "the partner has read the previous pass",
        // the second "the partner has written this pass".
        char* xb = xbuf + (size_t)b * (2 * R * 3 * LB_ROW);
        row_barrier(1 + b, 64);
#pragma unroll
        for (int r = 0; r < R; r++) {
            if (r < nact) {
                char* give = xb + (size_t)((1 - P) * R + r) * (3 * LB_ROW) + j * 16;   // read by the partner (warp 1 - P)
#pragma unroll
                for (int k = 0; k < 3; k++)
                    *reinterpret_cast<float4*>(give + k * LB_ROW) = make_float4(acc[r][12 * (1 - P) + 4 * k], acc[r][12 * (1 - P) + 4 * k + 1],
                                                                                 acc[r][12 * (1 - P) + 4 * k + 2], acc[r][12 * (1 - P) + 4 * k + 3]);
            }
        }
        row_barrier(1 + b, 64);
#pragma unroll
        for (int r = 0; r < R; r++) {
            if (r >= nact) break;
            float sum[12];
            const char* take = xb + (size_t)(P * R + r) * (3 * LB_ROW) + j * 16;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const float4 v = *reinterpret_cast<const float4*>(take + k * LB_ROW);
                // (x, y directions) + (z, t directions); IEEE addition commutes, so both warps add the same way
                const float* mine = acc[r] + 12 * P + 4 * k;
                const f2 s0 = add2(pk(mine[0], mine[1]), pk(v.x, v.y)), s1 = add2(pk(mine[2], mine[3]), pk(v.z, v.w));
                upk(s0, sum[4 * k], sum[4 * k + 1]);
                upk(s1, sum[4 * k + 2], sum[4 * k + 3]);
            }

            // epilogue on the 6 complex numbers of this half: o = Td (D in) [+ Tx x]
            float o[12];
            if (d_real) cscale_real_f32<6>(cdr, sum, o);   // Td real (-kappa^2): the same values without the zero products
            else cscale_f32<6>(cdr, cdi, sum, o);
            if (XPAY) caxpy_f32<6>(cxr, cxi, xv[r], o);
            double nrm = 0.0;
            if (EPI == EPI_RESID) {   // r -= alpha q, |r|^2 (q itself is never stored)
                const float alpha = (float)a.cg->alpha[src + r];
                raxpy_f32<6>(-alpha, o, rv[r]);
#pragma unroll
                for (int k = 0; k < 12; k++) o[k] = rv[r][k];
            }
            if (EPI != EPI_NONE) {   // two packed fp32 chains of six squares each, then fp64 (as norm2_site)
#pragma unroll
                for (int h2 = 0; h2 < 2; h2++) {
                    f2 pz = mul2(pk(o[6 * h2], o[6 * h2 + 1]), pk(o[6 * h2], o[6 * h2 + 1]));
                    pz = fma2(pk(o[6 * h2 + 2], o[6 * h2 + 3]), pk(o[6 * h2 + 2], o[6 * h2 + 3]), pz);
                    pz = fma2(pk(o[6 * h2 + 4], o[6 * h2 + 5]), pk(o[6 * h2 + 4], o[6 * h2 + 5]), pz);
                    float pa, pb;
                    upk(pz, pa, pb);
                    nrm += (double)(pa + pb);
                }
            }
#pragma unroll
            for (int k = 0; k < 3; k++)
                *reinterpret_cast<float4*>(a.out + o_site + r * fb + k * LB_ROW) = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
            if (EPI != EPI_NONE) {   // one partial per (source, tile, warp): 32 sites x 12 reals, fixed shuffle tree
                const double v = warp_sum(nrm);
                if (j == 0) a.partials[((size_t)(src + r) * bg.ntiles + tile) * 8 + w] = v;
            }
        }

        it += nact;
        if (last_pass) { src = 0; tile += gridDim.x; }
        else src += nact;
    }
}

template <int RECON, bool DAGGER, bool XPAY, int EPI>
__global__ void __launch_bounds__(BTHREADS, 1)
k_dslash_box(const __grid_constant__ BoxMaps maps, const BoxArgs a)
{
    extern __shared__ __align__(1024) char smem[];
    __shared__ __align__(8) uint64_t full[NST_MAX];
    __shared__ unsigned ticket[NST_MAX];
    if (a.check_done && a.cg->all_done) return;
    const BoxGeom& bg = a.bg;
    const int NST = bg.nst;
    char* xbuf = smem + (size_t)NST * bg.stage_bytes;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; s++) { mbar_init(&full[s], 1); ticket[s] = 0; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {   // prologue: the first NST (tile, source) pairs of this CTA
        const int my_tiles = ((int)blockIdx.x < bg.ntiles) ? (bg.ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
        const int n_iter = my_tiles * a.nrhs;
        int src = 0, tile = blockIdx.x;
        for (int it = 0; it < NST && it < n_iter; it++) {
            issue_stage(bg, maps, smem + (size_t)it * bg.stage_bytes, &full[it], tile, src);
            if (++src == a.nrhs) { src = 0; tile += gridDim.x; }
        }
    }
    if (((threadIdx.x >> 5) & 1) == 0) run_warp<RECON, DAGGER, XPAY, EPI, 0, BOX_R>(a, maps, smem, full, ticket, xbuf);
    else run_warp<RECON, DAGGER, XPAY, EPI, 1, BOX_R>(a, maps, smem, full, ticket, xbuf);
}

// ------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

bool box_geom(const Geom& g, BoxGeom& bg)
{
    const int Lxh = g.Lxh;
    if (Lxh < 1 || Lxh > 32 || (32 % Lxh) != 0) return false;
    const int rpb = 32 / Lxh;
    if (g.L[1] % rpb != 0 || (g.L[2] & 1) || (g.L[3] & 1)) return false;
    bg.Lxh = Lxh;
    bg.lxs = 0;
    while ((1 << bg.lxs) < Lxh) bg.lxs++;
    bg.rpb = rpb;
    bg.nyb = g.L[1] / rpb;
    bg.Lz = g.L[2];
    bg.Lt = g.L[3];
    bg.Lzh = g.L[2] / 2;
    bg.Lth = g.L[3] / 2;
    bg.HB = NCH32 * Lxh * 16;
    if (bg.HB % 128 != 0) return false;   // TMA destinations are 128-byte aligned
    bg.stage_bytes = 12 * CB + 8 * bg.HB;
    bg.nst = NST_MAX;
    while (bg.nst > 2 && (size_t)bg.nst * bg.stage_bytes + XBUF_BYTES > SMEM_MAX) bg.nst--;
    bg.ntiles = bg.nyb * bg.Lzh * bg.Lth;
    bg.Zs = 1;
    for (int z = 1; z <= 4 && z <= bg.Lzh; z++)
        if (bg.Lzh % z == 0) bg.Zs = z;
    bg.d_nyb = make_fastdiv(bg.nyb);
    bg.d_Zs = make_fastdiv(bg.Zs);
    bg.d_Lth = make_fastdiv(bg.Lth);
    return true;
}

// the four tensor maps of an fp32 single-parity field of nrhs sources starting at `field`
int make_maps(tsm_ctx* ctx, const BoxGeom& bg, const void* field, int nrhs, BoxMaps& m)
{
    for (const BoxMapCache& c : ctx->box_maps)
        if (c.field == field && c.nrhs == nrhs) { memcpy(&m, c.maps, sizeof(BoxMaps)); return TSM_OK; }
    EncodeTiledFn enc = encode_fn();
    if (!enc) return tsm_fail(ctx, TSM_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const cuuint64_t dims[5] = {128, (cuuint64_t)NCH32, (cuuint64_t)bg.nyb, (cuuint64_t)bg.Lz, (cuuint64_t)bg.Lt * nrhs};
    const cuuint64_t strides[4] = {LB_ROW, (cuuint64_t)CB, (cuuint64_t)CB * bg.nyb, (cuuint64_t)CB * bg.nyb * bg.Lz};
    const cuuint32_t es[5] = {1, 1, 1, 1, 1};
    const cuuint32_t boxes[4][5] = {{128, NCH32, 1, 2, 2}, {(cuuint32_t)bg.Lxh * 4, NCH32, 1, 2, 2}, {128, NCH32, 1, 1, 2}, {128, NCH32, 1, 2, 1}};
    CUtensorMap* out[4] = {&m.center, &m.yrow, &m.zface, &m.tface};
    for (int k = 0; k < 4; k++) {
        const CUresult r = enc(out[k], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<void*>(field), dims, strides, boxes[k], es,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return tsm_fail(ctx, TSM_ECUDA, "cuTensorMapEncodeTiled failed");
    }
    if (ctx->box_maps.size() >= 64) ctx->box_maps.erase(ctx->box_maps.begin());
    BoxMapCache c;
    c.field = field;
    c.nrhs = nrhs;
    static_assert(sizeof(c.maps) == sizeof(BoxMaps), "cache entry size");
    memcpy(c.maps, &m, sizeof(BoxMaps));
    ctx->box_maps.push_back(c);
    return TSM_OK;
}

template <int RECON, bool DAGGER, bool XPAY, int EPI>
int launch_box_t(tsm_ctx* ctx, const BoxGeom& bg, const BoxMaps& maps, const BoxArgs& a)
{
    const size_t smem = (size_t)bg.nst * bg.stage_bytes + XBUF_BYTES;   // stage ring + exchange buffers
    auto kern = k_dslash_box<RECON, DAGGER, XPAY, EPI>;
    static unsigned long long attr_done = 0;   // per device
    if (!((attr_done >> (ctx->device & 63)) & 1ull)) {
        TSM_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
        attr_done |= 1ull << (ctx->device & 63);
    }
    int grid = ctx->nsm;
    if (grid > bg.ntiles) grid = bg.ntiles;
    const int pi = prof_begin(ctx, TSM_F32, EPI == EPI_RESID ? 3 : (EPI == EPI_NORM ? 2 : (XPAY ? 1 : 0)), a.nrhs);
    kern<<<grid, BTHREADS, smem, ctx->stream>>>(maps, a);
    prof_end(ctx, pi);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

template <int RECON>
int launch_box_v(tsm_ctx* ctx, const BoxGeom& bg, const BoxMaps& maps, const BoxArgs& a, bool dagger, bool xpay, int epi)
{
#define GO(DG, XP, EP) return launch_box_t<RECON, DG, XP, EP>(ctx, bg, maps, a)
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

// Can this context's fp32 stencils run on the box kernel (lattice shape and enough shared memory)?
bool box_stencil_supported(const tsm_ctx* ctx)
{
    BoxGeom bg;
    if (!box_geom(ctx->g, bg)) return false;
    return (size_t)bg.nst * bg.stage_bytes + XBUF_BYTES <= SMEM_MAX && encode_fn() != nullptr;
}

int launch_dslash_box(tsm_ctx* ctx, int out_parity, bool dagger, int nrhs, const void* in, const void* x, void* out,
                      const DslashCoef& c, int mode)
{
    BoxGeom bg;
    if (!box_geom(ctx->g, bg)) return tsm_fail(ctx, TSM_ESTATE, "box stencil: unsupported lattice shape");
    const int chk = (mode >> 1) & 1, epi = (mode & 4) ? EPI_RESID : ((mode & 1) ? EPI_NORM : EPI_NONE);
    if (epi != EPI_NONE && (size_t)bg.ntiles * 8 * nrhs > ctx->norm_partials_count) return tsm_fail(ctx, TSM_ESTATE, "reduction scratch too small");
    BoxMaps maps;
    int rc = make_maps(ctx, bg, in, nrhs, maps);
    if (rc) return rc;
    BoxArgs a;
    a.bg = bg;
    a.par = out_parity;
    a.nrhs = nrhs;
    a.theta = ctx->g.theta;
    a.check_done = chk;
    a.pack = (const char*)ctx->gauge32[out_parity];
    a.x = (const char*)x;
    a.out = (char*)out;
    a.cf = c;
    a.partials = ctx->norm_partials;
    a.cg = ctx->cg;
    ctx->norm_ntiles = bg.ntiles * 8;
    ctx->norm_reduced = false;
    if (ctx->recon == 18) return launch_box_v<18>(ctx, bg, maps, a, dagger, x != nullptr, epi);
    return launch_box_v<12>(ctx, bg, maps, a, dagger, x != nullptr, epi);
}
