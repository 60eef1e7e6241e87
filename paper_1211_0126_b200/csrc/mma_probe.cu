// mma_probe.cu -- the tensor-core question of north_star, settled by a measurement.
//
// north_star keeps tensor cores off "unless a multi-RHS SU(3) x (3 x N_rhs) tile is shown by ncu to be a profitable
// dense contraction".  The only dense contraction of the stencil is, per site and hop, G = U H with U one 3 x 3
// complex link and H the 3 x (2 N) block of the N sources' projected half spinors (N = 12: 24 columns) -- in real
// arithmetic a (6 x 6) x (6 x 24) product whose left factor changes with every site and hop.  This file times that
// product, and nothing else, in the formulations that exist on sm_100a for operands living in registers:
//   variant 0: packed fp32 FMAs (FFMA2), one thread per (site, source), the stencil's own su3_mul
//   variant 1: mma.sync m16n8k8 TF32, one MMA per 8 columns (TF32 rounding of both operands: breaks the 1e-5 parity bar)
//   variant 2: 3xTF32 (big/small split of both operands; A_big and A_small stacked in the 16 rows of one MMA, so
//              two MMAs per 8 columns instead of three): holds fp32 accuracy
//   variant 3: fp64 FMAs (DFMA), one thread per (site, source)
//   variant 4: fp64 mma.sync m8n8k4 (DMMA), two k-steps x three 8-column tiles per (site, hop)
// Every variant loads its operands once into registers, in the fragment layout that suits it (so the tensor path is
// NOT charged for the lane shuffles a real stencil would need to turn gathered spinors into B fragments), and then
// repeats the product INNER times on H + it * eps, accumulating G: the probe measures the issue rate of the
// arithmetic alone.  tcgen05.mma needs both operands as shared-memory / TMEM
// tiles with M >= 64 rows that SHARE the right factor, which a per-site 6 x 6 left factor cannot provide, so mma.sync
// is the only tensor path there is for this product.  Results go to profiles/r02_mma_experiment.md (bench.py --probe-mma).
#include <cstdint>

#include "dslash_common.cuh"

namespace {

constexpr int NCOL = 24;   // 12 sources x 2 spin rows of the projected half spinor

__device__ __forceinline__ float hash_unit(uint32_t a, uint32_t b)
{
    uint32_t x = a * 0x9E3779B9u ^ (b + 0x7F4A7C15u) * 0x85EBCA6Bu;
    x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
    return (float)(x >> 8) * (1.0f / 8388608.0f) - 1.0f;   // [-1, 1)
}

// U[site][18] (row-major complex 3 x 3), H[site][col][6] = (c0.re, c0.im, c1.re, c1.im, c2.re, c2.im), both fp32 values
// (the fp64 variants read the same numbers widened), ref[site][col][6] = sum_it U (H + it eps) in fp64
constexpr float PROBE_EPS = 1.0f / 1024.0f;
__global__ void k_probe_fill(const int nsites, const int inner, float* U, float* H, double* ref)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsites) return;
    float u[18];
    for (int k = 0; k < 18; k++) { u[k] = 0.6f * hash_unit(s, k); U[(size_t)s * 18 + k] = u[k]; }
    for (int c = 0; c < NCOL; c++) {
        float h[6];
        for (int k = 0; k < 6; k++) { h[k] = hash_unit(s + 0x51ED27, c * 6 + k); H[((size_t)s * NCOL + c) * 6 + k] = h[k]; }
        double hs[6];   // sum over it of (h + it eps)
        for (int k = 0; k < 6; k++) hs[k] = (double)inner * h[k] + (double)PROBE_EPS * 0.5 * inner * (inner - 1);
        for (int r = 0; r < 3; r++) {
            double re = 0, im = 0;
            for (int k = 0; k < 3; k++) {
                re += (double)u[6 * r + 2 * k] * hs[2 * k] - (double)u[6 * r + 2 * k + 1] * hs[2 * k + 1];
                im += (double)u[6 * r + 2 * k] * hs[2 * k + 1] + (double)u[6 * r + 2 * k + 1] * hs[2 * k];
            }
            ref[((size_t)s * NCOL + c) * 6 + 2 * r] = re;
            ref[((size_t)s * NCOL + c) * 6 + 2 * r + 1] = im;
        }
    }
}

// variants 0 and 3: one thread per (site, source): both spin rows of that source
template <typename T> __global__ void __launch_bounds__(384) k_probe_fma(const int nsites, const int inner, const float* __restrict__ U, const float* __restrict__ H, T* __restrict__ G)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int s = idx / 12, src = idx - s * 12;
    if (s >= nsites) return;
    T u[18], h[12], acc[12];
#pragma unroll
    for (int k = 0; k < 18; k++) u[k] = (T)__ldg(U + (size_t)s * 18 + k);
#pragma unroll
    for (int k = 0; k < 12; k++) { h[k] = (T)__ldg(H + ((size_t)s * NCOL + 2 * src) * 6 + k); acc[k] = 0; }
    for (int it = 0; it < inner; it++) {
        T o[12];
        su3_mul(u, h, o);
        su3_mul(u, h + 6, o + 6);
#pragma unroll
        for (int k = 0; k < 12; k++) { acc[k] += o[k]; h[k] += (T)PROBE_EPS; }
    }
#pragma unroll
    for (int k = 0; k < 12; k++) G[((size_t)s * NCOL + 2 * src) * 6 + k] = acc[k];
}

__device__ __forceinline__ uint32_t to_tf32(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void mma_tf32(float* d, const uint32_t* a, const uint32_t* b)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// real 6 x 6 form of the link: rows 0-2 = (Re U, -Im U), rows 3-5 = (Im U, Re U); k = (re c0..c2, im c0..c2)
__device__ __forceinline__ float link_real(const float* __restrict__ u, int r, int k)
{
    if (r >= 6 || k >= 6) return 0.f;
    const int rr = r % 3, kk = k % 3;
    const float re = __ldg(u + 6 * rr + 2 * kk), im = __ldg(u + 6 * rr + 2 * kk + 1);
    return (r < 3) == (k < 3) ? re : (r < 3 ? -im : im);
}

// variants 1 and 2: one warp per site at a time.  A fragment (m16n8k8, row major): a0 (row g, col t), a1 (row g + 8,
// col t), a2 (row g, col t + 4), a3 (row g + 8, col t + 4), g = lane / 4, t = lane % 4.  B fragment: b0 (k = t, n = g),
// b1 (k = t + 4, n = g).  C: c0, c1 (row g, cols 2t, 2t + 1), c2, c3 (row g + 8, same cols).
template <bool SPLIT> __global__ void __launch_bounds__(256) k_probe_tf32(const int nsites, const int inner, const float* __restrict__ U, const float* __restrict__ H, float* __restrict__ G)
{
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int s = warp; s < nsites; s += nwarps) {
        const float* u = U + (size_t)s * 18;
        const float a_lo = link_real(u, g, t), a_hi = link_real(u, g, t + 4);
        uint32_t A1[4], A2[4];
        A1[0] = to_tf32(a_lo); A1[2] = to_tf32(a_hi);
        if (SPLIT) {   // rows 8-13 of the first MMA carry the small parts of A
            A1[1] = to_tf32(a_lo - __uint_as_float(A1[0])); A1[3] = to_tf32(a_hi - __uint_as_float(A1[2]));
            A2[0] = A1[0]; A2[2] = A1[2]; A2[1] = 0; A2[3] = 0;
        } else {
            A1[1] = 0; A1[3] = 0;
        }
        float b_lo[3], b_hi[3], c[3][4];
#pragma unroll
        for (int nt = 0; nt < 3; nt++) {
            // column n = 8 nt + g of H; k index -> (re c, im c): k < 3: re of colour k, else im of colour k - 3
            const float* h = H + ((size_t)s * NCOL + 8 * nt + g) * 6;
            b_lo[nt] = t < 3 ? __ldg(h + 2 * t) : __ldg(h + 1);          // k = t:     re c_t, or (t = 3) im c0
            b_hi[nt] = t < 2 ? __ldg(h + 2 * (t + 1) + 1) : 0.f;         // k = t + 4: im c_{t+1} (k = 4, 5), 0 for k = 6, 7
#pragma unroll
            for (int k = 0; k < 4; k++) c[nt][k] = 0.f;
        }
        const float eps_hi = t < 2 ? PROBE_EPS : 0.f;
        for (int it = 0; it < inner; it++) {
#pragma unroll
            for (int nt = 0; nt < 3; nt++) {
                uint32_t B1[2] = {to_tf32(b_lo[nt]), to_tf32(b_hi[nt])};
                mma_tf32(c[nt], A1, B1);
                if (SPLIT) {
                    uint32_t B2[2] = {to_tf32(b_lo[nt] - __uint_as_float(B1[0])), to_tf32(b_hi[nt] - __uint_as_float(B1[1]))};
                    mma_tf32(c[nt], A2, B2);
                }
                b_lo[nt] += PROBE_EPS;
                b_hi[nt] += eps_hi;
            }
        }
#pragma unroll
        for (int nt = 0; nt < 3; nt++) {
            if (SPLIT) { c[nt][0] += c[nt][2]; c[nt][1] += c[nt][3]; }
            // row g of G_real (g < 6): g < 3 -> re of colour g, else im of colour g - 3; columns 8 nt + 2t, 2t + 1
            if (g < 6) {
                const int comp = g < 3 ? 2 * g : 2 * (g - 3) + 1;
                G[((size_t)s * NCOL + 8 * nt + 2 * t) * 6 + comp] = c[nt][0];
                G[((size_t)s * NCOL + 8 * nt + 2 * t + 1) * 6 + comp] = c[nt][1];
            }
        }
    }
}

// variant 4: fp64 m8n8k4.  A (8 x 4): a0 (row g, col t).  B (4 x 8): b0 (k = t, n = g).  C (8 x 8): c0, c1 (row g, cols 2t, 2t+1).
__global__ void __launch_bounds__(256) k_probe_dmma(const int nsites, const int inner, const float* __restrict__ U, const float* __restrict__ H, double* __restrict__ G)
{
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int s = warp; s < nsites; s += nwarps) {
        const float* u = U + (size_t)s * 18;
        const double a0 = (double)link_real(u, g, t), a1 = (double)link_real(u, g, t + 4);
        double b0[3], b1[3], c0[3], c1[3];
#pragma unroll
        for (int nt = 0; nt < 3; nt++) {
            const float* h = H + ((size_t)s * NCOL + 8 * nt + g) * 6;
            b0[nt] = (double)(t < 3 ? __ldg(h + 2 * t) : __ldg(h + 1));
            b1[nt] = (double)(t < 2 ? __ldg(h + 2 * (t + 1) + 1) : 0.f);
            c0[nt] = 0; c1[nt] = 0;
        }
        const double eps_hi = t < 2 ? (double)PROBE_EPS : 0.0;
        for (int it = 0; it < inner; it++) {
#pragma unroll
            for (int nt = 0; nt < 3; nt++) {
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0[nt]), "+d"(c1[nt]) : "d"(a0), "d"(b0[nt]));
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0[nt]), "+d"(c1[nt]) : "d"(a1), "d"(b1[nt]));
                b0[nt] += (double)PROBE_EPS;
                b1[nt] += eps_hi;
            }
        }
#pragma unroll
        for (int nt = 0; nt < 3; nt++)
            if (g < 6) {
                const int comp = g < 3 ? 2 * g : 2 * (g - 3) + 1;
                G[((size_t)s * NCOL + 8 * nt + 2 * t) * 6 + comp] = c0[nt];
                G[((size_t)s * NCOL + 8 * nt + 2 * t + 1) * 6 + comp] = c1[nt];
            }
    }
}

template <typename T> __global__ void k_probe_err(const size_t n, const T* __restrict__ G, const double* __restrict__ ref, double* out)
{
    // max |G - ref| and max |ref| over the array, by one block (the probe arrays are small)
    __shared__ double sm[2][256];
    double e = 0, m = 0;
    for (size_t k = threadIdx.x; k < n; k += blockDim.x) {
        e = fmax(e, fabs((double)G[k] - ref[k]));
        m = fmax(m, fabs(ref[k]));
    }
    sm[0][threadIdx.x] = e; sm[1][threadIdx.x] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 256; k++) { e = fmax(e, sm[0][k]); m = fmax(m, sm[1][k]); }
        out[0] = e; out[1] = m;
    }
}

}  // namespace

extern "C" int tsm_probe_su3_tensor(tsm_ctx* ctx, int variant, int nsites, int inner, int reps, double* us_per_launch, double* max_rel_err)
{
    int rc = ctx_enter(ctx, false, false, false);
    if (rc) return rc;
    if (variant < 0 || variant > 4 || nsites < 1 || nsites > (1 << 22) || inner < 1 || inner > 4096 || reps < 1 || !us_per_launch || !max_rel_err)
        return tsm_fail(ctx, TSM_EINVAL, "bad probe arguments");
    float *U = nullptr, *H = nullptr;
    double *ref = nullptr, *errbuf = nullptr;
    void* G = nullptr;
    const size_t nG = (size_t)nsites * NCOL * 6;
    const bool f64 = variant >= 3;
    TSM_CUDA(ctx, cudaMalloc(&U, (size_t)nsites * 18 * sizeof(float)));
    TSM_CUDA(ctx, cudaMalloc(&H, nG * sizeof(float)));
    TSM_CUDA(ctx, cudaMalloc(&ref, nG * sizeof(double)));
    TSM_CUDA(ctx, cudaMalloc(&G, nG * (f64 ? 8 : 4)));
    TSM_CUDA(ctx, cudaMalloc(&errbuf, 2 * sizeof(double)));
    k_probe_fill<<<(nsites + 127) / 128, 128, 0, ctx->stream>>>(nsites, inner, U, H, ref);
    auto launch = [&]() {
        const int nthreads_fma = nsites * 12;
        const int grid_w = ctx->nsm * 8;   // warp-per-site variants: persistent, 8 x 8 warps per SM
        switch (variant) {
            case 0: k_probe_fma<float><<<(nthreads_fma + 383) / 384, 384, 0, ctx->stream>>>(nsites, inner, U, H, (float*)G); break;
            case 1: k_probe_tf32<false><<<grid_w, 256, 0, ctx->stream>>>(nsites, inner, U, H, (float*)G); break;
            case 2: k_probe_tf32<true><<<grid_w, 256, 0, ctx->stream>>>(nsites, inner, U, H, (float*)G); break;
            case 3: k_probe_fma<double><<<(nthreads_fma + 383) / 384, 384, 0, ctx->stream>>>(nsites, inner, U, H, (double*)G); break;
            default: k_probe_dmma<<<grid_w, 256, 0, ctx->stream>>>(nsites, inner, U, H, (double*)G); break;
        }
    };
    for (int k = 0; k < 3; k++) launch();
    TSM_CUDA(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
    for (int k = 0; k < reps; k++) launch();
    TSM_CUDA(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->launches += reps + 4;
    if (f64) k_probe_err<double><<<1, 256, 0, ctx->stream>>>(nG, (const double*)G, ref, errbuf);
    else k_probe_err<float><<<1, 256, 0, ctx->stream>>>(nG, (const float*)G, ref, errbuf);
    double host[2] = {0, 0};
    TSM_CUDA(ctx, cudaMemcpyAsync(host, errbuf, sizeof(host), cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    float ms = 0;
    TSM_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    *us_per_launch = (double)ms * 1e3 / reps;
    *max_rel_err = host[1] > 0 ? host[0] / host[1] : 0.0;
    cudaFree(U); cudaFree(H); cudaFree(ref); cudaFree(G); cudaFree(errbuf);
    TSM_CUDA(ctx, cudaGetLastError());
    return TSM_OK;
}
