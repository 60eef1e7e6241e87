// fields.cu -- H1-H3: layout conversion (host lex fp64 <-> native even/odd vectorised fields),
// gauge ingest into per-parity link packs, the counter-based Z4/Z2 noise kernel, and the
// site-diagonal twist / precision-conversion kernels.
#include "tsm_internal.cuh"

namespace {

__device__ __forceinline__ void atomic_max_nonneg(double* addr, double v)
{
    // non-negative doubles order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

// max that keeps a NaN operand (fmax drops it: a link full of NaN would report deviation 0)
__device__ __forceinline__ double max_nan(double a, double b) { return (a != a || b != b) ? __longlong_as_double(0x7ff8000000000000LL) : (a > b ? a : b); }

// |U^dag U - 1|_max and |det U - 1| of one row-major complex 3x3 matrix (18 doubles)
__device__ double unitarity_dev(const double* u)
{
    double dev = 0;
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) {
            double re = (a == b) ? -1.0 : 0.0, im = 0;
            for (int k = 0; k < 3; k++) {   // sum_k conj(U_ka) U_kb
                const double ar = u[2 * (3 * k + a)], ai = u[2 * (3 * k + a) + 1];
                const double br = u[2 * (3 * k + b)], bi = u[2 * (3 * k + b) + 1];
                re += ar * br + ai * bi;
                im += ar * bi - ai * br;
            }
            dev = max_nan(dev, max_nan(fabs(re), fabs(im)));
        }
    double dr = 0, di = 0;
    for (int c = 0; c < 3; c++) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        // cofactor of U_0c: U_1a U_2b - U_1b U_2a
        const double cr = (u[2 * (3 + a)] * u[2 * (6 + b)] - u[2 * (3 + a) + 1] * u[2 * (6 + b) + 1]) -
                          (u[2 * (3 + b)] * u[2 * (6 + a)] - u[2 * (3 + b) + 1] * u[2 * (6 + a) + 1]);
        const double ci = (u[2 * (3 + a)] * u[2 * (6 + b) + 1] + u[2 * (3 + a) + 1] * u[2 * (6 + b)]) -
                          (u[2 * (3 + b)] * u[2 * (6 + a) + 1] + u[2 * (3 + b) + 1] * u[2 * (6 + a)]);
        dr += u[2 * c] * cr - u[2 * c + 1] * ci;
        di += u[2 * c] * ci + u[2 * c + 1] * cr;
    }
    return max_nan(dev, max_nan(fabs(dr - 1.0), fabs(di)));
}

// raw: [4][V][3][3][2] fp64 in lex order.  One thread per (parity, cb site): writes its 8 links
// into the fp64 pack and the fp32 pack (18 or 12 reals).
__global__ void k_gauge_pack(const Geom g, const int recon, const double* __restrict__ raw, void* pack64_0, void* pack64_1,
                             void* pack32_0, void* pack32_1, double* max_dev)
{
    const int Vh = g.Vh;
    double dev = 0;
    for (int tid = blockIdx.x * blockDim.x + threadIdx.x; tid < 2 * Vh; tid += gridDim.x * blockDim.x) {
        const int par = tid / Vh, i = tid - par * Vh;
        const SiteCoord s = decode_site(g, i, par);
        const long long lex = lex_of_site(g, s);
        const int x[4] = {2 * s.xh + s.rowpar, s.y, s.z, s.t};
        char* p64 = pack64_0 ? site_ptr<72>(par ? pack64_1 : pack64_0, i) : nullptr;   // no fp64 pack in a low-precision-only workspace
        char* p32 = recon == 18 ? site_ptr<36>(par ? pack32_1 : pack32_0, i) : site_ptr<24>(par ? pack32_1 : pack32_0, i);
        for (int mu = 0; mu < 4; mu++) {
            int xm[4] = {x[0], x[1], x[2], x[3]};
            xm[mu] = (x[mu] + g.L[mu] - 1) % g.L[mu];
            const long long lexm = xm[0] + (long long)g.L[0] * (xm[1] + (long long)g.L[1] * (xm[2] + (long long)g.L[2] * xm[3]));
            const double* uf = raw + ((size_t)mu * g.V + lex) * 18;
            const double* um = raw + ((size_t)mu * g.V + lexm) * 18;
            double f[18], b[18];
            for (int k = 0; k < 18; k++) f[k] = uf[k];
            for (int r = 0; r < 3; r++)
                for (int c = 0; c < 3; c++) {   // b = um^dagger
                    b[2 * (3 * r + c)] = um[2 * (3 * c + r)];
                    b[2 * (3 * r + c) + 1] = -um[2 * (3 * c + r) + 1];
                }
            dev = max_nan(dev, unitarity_dev(f));
            if (p64)
                for (int j = 0; j < 9; j++) {
                    *reinterpret_cast<double2*>(p64 + (18 * mu + j) * LB_ROW) = make_double2(f[2 * j], f[2 * j + 1]);
                    *reinterpret_cast<double2*>(p64 + (18 * mu + 9 + j) * LB_ROW) = make_double2(b[2 * j], b[2 * j + 1]);
                }
            if (recon == 18) {
                float l[36];
                for (int k = 0; k < 18; k++) { l[k] = (float)f[k]; l[18 + k] = (float)b[k]; }
                for (int j = 0; j < 9; j++)
                    *reinterpret_cast<float4*>(p32 + (9 * mu + j) * LB_ROW) = make_float4(l[4 * j], l[4 * j + 1], l[4 * j + 2], l[4 * j + 3]);
            } else {
                for (int j = 0; j < 3; j++) {
                    *reinterpret_cast<float4*>(p32 + (6 * mu + j) * LB_ROW) = make_float4((float)f[4 * j], (float)f[4 * j + 1], (float)f[4 * j + 2], (float)f[4 * j + 3]);
                    *reinterpret_cast<float4*>(p32 + (6 * mu + 3 + j) * LB_ROW) = make_float4((float)b[4 * j], (float)b[4 * j + 1], (float)b[4 * j + 2], (float)b[4 * j + 3]);
                }
            }
        }
    }
    atomic_max_nonneg(max_dev, dev);
}

template <int PREC>
__global__ void k_pack_spinor(const Geom g, const int nrhs, const size_t par_stride, const double* __restrict__ lexf, void* native)
{
    using T = typename PT<PREC>::real;
    const int Vh = g.Vh;
    const long long n = 2LL * Vh * nrhs;
    for (long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x; tid < n; tid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(tid % Vh);
        const int rhs = (int)((tid / Vh) % nrhs);
        const int par = (int)(tid / ((long long)Vh * nrhs));
        const SiteCoord s = decode_site(g, i, par);
        const double* src = lexf + ((size_t)rhs * g.V + lex_of_site(g, s)) * 24;
        T v[24];
#pragma unroll
        for (int k = 0; k < 24; k++) v[k] = (T)src[k];
        char* dst = (char*)native + par_stride * par + field_bytes(PREC, Vh, 1) * rhs;
        store_spinor<PREC>(dst, i, v);
    }
}

template <int PREC>
__global__ void k_unpack_spinor(const Geom g, const int nrhs, const size_t par_stride, const void* __restrict__ native, double* lexf)
{
    using T = typename PT<PREC>::real;
    const int Vh = g.Vh;
    const long long n = 2LL * Vh * nrhs;
    for (long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x; tid < n; tid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(tid % Vh);
        const int rhs = (int)((tid / Vh) % nrhs);
        const int par = (int)(tid / ((long long)Vh * nrhs));
        const SiteCoord s = decode_site(g, i, par);
        const char* src = (const char*)native + par_stride * par + field_bytes(PREC, Vh, 1) * rhs;
        T v[24];
        load_spinor<PREC>(src, i, v);
        double* dst = lexf + ((size_t)rhs * g.V + lex_of_site(g, s)) * 24;
#pragma unroll
        for (int k = 0; k < 24; k++) dst[k] = (double)v[k];
    }
}

// H3: eta_j(x, alpha, c) straight into a full-lattice native field [parity][rhs][chunk][cb].
template <int PREC>
__global__ void k_noise(const Geom g, const int nrhs, const uint64_t seed, const uint32_t* __restrict__ ids, const int kind, void* native)
{
    using T = typename PT<PREC>::real;
    const int Vh = g.Vh;
    const long long n = 2LL * Vh * nrhs;
    for (long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x; tid < n; tid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(tid % Vh);
        const int rhs = (int)((tid / Vh) % nrhs);
        const int par = (int)(tid / ((long long)Vh * nrhs));
        const SiteCoord s = decode_site(g, i, par);
        const uint32_t bits = noise_bits(lex_of_site(g, s), seed, ids[rhs], kind);
        T v[24];
#pragma unroll
        for (int q = 0; q < 12; q++) {
            float re, im;
            noise_value((bits >> (2 * q)) & 3, kind, re, im);
            v[2 * q] = (T)re;
            v[2 * q + 1] = (T)im;
        }
        char* dst = (char*)native + field_bytes(PREC, Vh, nrhs) * par + field_bytes(PREC, Vh, 1) * rhs;
        store_spinor<PREC>(dst, i, v);
    }
}

// out = c (x) in on a single-parity field: c.up on spins 0,1, c.lo on spins 2,3.
template <int PREC>
__global__ void k_twist(const int Vh, const int nrhs, const void* __restrict__ in, void* out, const TwistCoef c)
{
    using T = typename PT<PREC>::real;
    const long long n = (long long)Vh * nrhs * 3;
    for (long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x; tid < n; tid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(tid % Vh);
        const int k8 = (int)((tid / Vh) % 3);
        const int rhs = (int)(tid / (3LL * Vh));
        const size_t off = field_bytes(PREC, Vh, 1) * rhs;
        T v[8], o[8];
        load8<PREC>((const char*)in + off, i, k8, v);
        twist8<T>(c, k8, v, o);
        store8<PREC>((char*)out + off, i, k8, o);
    }
}

template <int PIN, int POUT>
__global__ void k_convert(const int Vh, const int nfields, const void* __restrict__ in, void* out)
{
    const long long n = (long long)Vh * nfields * 3;
    for (long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x; tid < n; tid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(tid % Vh);
        const int k8 = (int)((tid / Vh) % 3);
        const int f = (int)(tid / (3LL * Vh));
        typename PT<PIN>::real v[8];
        typename PT<POUT>::real o[8];
        load8<PIN>((const char*)in + field_bytes(PIN, Vh, 1) * f, i, k8, v);
#pragma unroll
        for (int k = 0; k < 8; k++) o[k] = (typename PT<POUT>::real)v[k];
        store8<POUT>((char*)out + field_bytes(POUT, Vh, 1) * f, i, k8, o);
    }
}

inline int grid_for(const tsm_ctx* ctx, long long n, int bs)
{
    long long gx = (n + bs - 1) / bs;
    const long long cap = (long long)ctx->nsm * 16;
    return (int)(gx > cap ? cap : (gx < 1 ? 1 : gx));
}

}  // namespace

int launch_gauge_pack(tsm_ctx* ctx, double* max_dev_out)
{
    TSM_CUDA(ctx, cudaMemsetAsync(max_dev_out, 0, sizeof(double), ctx->stream));
    k_gauge_pack<<<grid_for(ctx, 2LL * ctx->g.Vh, 128), 128, 0, ctx->stream>>>(
        ctx->g, ctx->recon, (const double*)ctx->staging, ctx->gauge64[0], ctx->gauge64[1], ctx->gauge32[0], ctx->gauge32[1], max_dev_out);
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

#define PREC_SWITCH(prec, CALL)                                          \
    switch (prec) {                                                      \
        case TSM_F64: { constexpr int P = TSM_F64; CALL; break; }        \
        case TSM_F32: { constexpr int P = TSM_F32; CALL; break; }        \
        case TSM_BF16: { constexpr int P = TSM_BF16; CALL; break; }      \
        default: return tsm_fail(ctx, TSM_EINVAL, "bad precision");      \
    }

// par_stride: bytes between the parity-0 and the parity-1 part of the native field (0: the dense [parity][rhs] field)
int launch_pack_spinor(tsm_ctx* ctx, int prec, int nrhs, const double* dev_lex, void* dev_native, size_t par_stride)
{
    const int gx = grid_for(ctx, 2LL * ctx->g.Vh * nrhs, 256);
    if (par_stride == 0) par_stride = field_bytes(prec, ctx->g.Vh, nrhs);
    PREC_SWITCH(prec, (k_pack_spinor<P><<<gx, 256, 0, ctx->stream>>>(ctx->g, nrhs, par_stride, dev_lex, dev_native)));
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_unpack_spinor(tsm_ctx* ctx, int prec, int nrhs, const void* dev_native, double* dev_lex, size_t par_stride)
{
    const int gx = grid_for(ctx, 2LL * ctx->g.Vh * nrhs, 256);
    if (par_stride == 0) par_stride = field_bytes(prec, ctx->g.Vh, nrhs);
    PREC_SWITCH(prec, (k_unpack_spinor<P><<<gx, 256, 0, ctx->stream>>>(ctx->g, nrhs, par_stride, dev_native, dev_lex)));
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_noise(tsm_ctx* ctx, int prec, int nrhs, uint64_t seed, const uint32_t* dev_ids, int kind, void* dev_full)
{
    const int gx = grid_for(ctx, 2LL * ctx->g.Vh * nrhs, 256);
    PREC_SWITCH(prec, (k_noise<P><<<gx, 256, 0, ctx->stream>>>(ctx->g, nrhs, seed, dev_ids, kind, dev_full)));
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_twist(tsm_ctx* ctx, int prec, int nrhs, const void* in, void* out, const TwistCoef& c)
{
    const int gx = grid_for(ctx, 3LL * ctx->g.Vh * nrhs, 256);
    PREC_SWITCH(prec, (k_twist<P><<<gx, 256, 0, ctx->stream>>>(ctx->g.Vh, nrhs, in, out, c)));
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}

int launch_convert(tsm_ctx* ctx, int prec_in, int prec_out, int nfields, const void* in, void* out)
{
    const int gx = grid_for(ctx, 3LL * ctx->g.Vh * nfields, 256);
    const int Vh = ctx->g.Vh;
#define CV(A, B) if (prec_in == A && prec_out == B) k_convert<A, B><<<gx, 256, 0, ctx->stream>>>(Vh, nfields, in, out); else
    CV(TSM_F64, TSM_F32) CV(TSM_F32, TSM_F64) CV(TSM_F32, TSM_BF16) CV(TSM_BF16, TSM_F32)
    CV(TSM_F64, TSM_BF16) CV(TSM_BF16, TSM_F64) CV(TSM_F64, TSM_F64) CV(TSM_F32, TSM_F32) CV(TSM_BF16, TSM_BF16)
        return tsm_fail(ctx, TSM_EINVAL, "bad precision");
#undef CV
    ctx->launches++;
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}
