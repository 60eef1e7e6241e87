// dslash_common.cuh -- spin projection / reconstruction shared by the stencil kernels (H5).
// gamma_mu = [[0, a_mu], [a_mu^dag, 0]] in the chiral basis C3: (1 +- gamma_mu) psi = [h; +- a_mu^dag h]
// with h = psi_up +- a_mu psi_low, so the SU(3) multiply acts on 2 spin x 3 colour only.
#pragma once
#include "packed_f32.cuh"
#include "tsm_internal.cuh"

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


// Sum of the 24 squares of a site's spinor for the fused norm / residual epilogues.  fp64 data: a plain fp64
// chain.  fp32 data: four fp32 partial sums of six squares each (FFMA chains), converted and added in fp64 --
// one quarter-rate F2F per partial instead of one per element (24 conversions per site cost ~10 % of the
// kernel); sums ACROSS sites stay fp64 with fixed trees (A19).  Both stencil kernels use this, so a source's
// partial sums are the same in any batch (A14).
template <typename T> __device__ __forceinline__ double norm2_site(const T* v)
{
    double s = 0.0;
    if constexpr (sizeof(T) == 8) {
#pragma unroll
        for (int k = 0; k < 24; k++) s += v[k] * v[k];
    } else {
#pragma unroll
        for (int j = 0; j < 4; j++) {   // six squares: a packed chain over three complex numbers, then re + im
            f2 p = mul2(pk(v[6 * j], v[6 * j + 1]), pk(v[6 * j], v[6 * j + 1]));
            p = fma2(pk(v[6 * j + 2], v[6 * j + 3]), pk(v[6 * j + 2], v[6 * j + 3]), p);
            p = fma2(pk(v[6 * j + 4], v[6 * j + 5]), pk(v[6 * j + 4], v[6 * j + 5]), p);
            float a, b;
            upk(p, a, b);
            s += (double)(a + b);
        }
    }
    return s;
}

// ------------------------------------------------------------------ fp32: the same operations on packed pairs
// Specialisations for float of project / accumulate and an overload of su3_mul: identical formulas, each complex
// add one FADD2, each complex multiply-add two FFMA2 (packed_f32.cuh).
template <int MU, int SGN> __device__ __forceinline__ void project_f32(const float* p, float* h)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const float p0r = p[2 * c], p0i = p[2 * c + 1], p1r = p[6 + 2 * c], p1i = p[6 + 2 * c + 1];
        const float p2r = p[12 + 2 * c], p2i = p[12 + 2 * c + 1], p3r = p[18 + 2 * c], p3i = p[18 + 2 * c + 1];
        f2 h0, h1;
        if (MU == 0) {          // h0 = p0 - i s p3, h1 = p1 - i s p2
            h0 = add2(pk(p0r, p0i), SGN > 0 ? c_mi(p3r, p3i) : c_i(p3r, p3i));
            h1 = add2(pk(p1r, p1i), SGN > 0 ? c_mi(p2r, p2i) : c_i(p2r, p2i));
        } else if (MU == 1) {   // h0 = p0 - s p3, h1 = p1 + s p2
            h0 = add2(pk(p0r, p0i), SGN > 0 ? c_neg(p3r, p3i) : c_pos(p3r, p3i));
            h1 = add2(pk(p1r, p1i), SGN > 0 ? c_pos(p2r, p2i) : c_neg(p2r, p2i));
        } else if (MU == 2) {   // h0 = p0 - i s p2, h1 = p1 + i s p3
            h0 = add2(pk(p0r, p0i), SGN > 0 ? c_mi(p2r, p2i) : c_i(p2r, p2i));
            h1 = add2(pk(p1r, p1i), SGN > 0 ? c_i(p3r, p3i) : c_mi(p3r, p3i));
        } else {                // h0 = p0 + s p2, h1 = p1 + s p3
            h0 = add2(pk(p0r, p0i), SGN > 0 ? c_pos(p2r, p2i) : c_neg(p2r, p2i));
            h1 = add2(pk(p1r, p1i), SGN > 0 ? c_pos(p3r, p3i) : c_neg(p3r, p3i));
        }
        upk(h0, h[2 * c], h[2 * c + 1]);
        upk(h1, h[6 + 2 * c], h[6 + 2 * c + 1]);
    }
}
template <> __device__ __forceinline__ void project<float, 0, 1>(const float* p, float* h) { project_f32<0, 1>(p, h); }
template <> __device__ __forceinline__ void project<float, 0, -1>(const float* p, float* h) { project_f32<0, -1>(p, h); }
template <> __device__ __forceinline__ void project<float, 1, 1>(const float* p, float* h) { project_f32<1, 1>(p, h); }
template <> __device__ __forceinline__ void project<float, 1, -1>(const float* p, float* h) { project_f32<1, -1>(p, h); }
template <> __device__ __forceinline__ void project<float, 2, 1>(const float* p, float* h) { project_f32<2, 1>(p, h); }
template <> __device__ __forceinline__ void project<float, 2, -1>(const float* p, float* h) { project_f32<2, -1>(p, h); }
template <> __device__ __forceinline__ void project<float, 3, 1>(const float* p, float* h) { project_f32<3, 1>(p, h); }
template <> __device__ __forceinline__ void project<float, 3, -1>(const float* p, float* h) { project_f32<3, -1>(p, h); }

template <int MU, int SGN> __device__ __forceinline__ void accumulate_f32(const float* g, float* acc)
{
#pragma unroll
    for (int q = 0; q < 6; q++) {   // acc_up += g
        const f2 a = add2(pk(acc[2 * q], acc[2 * q + 1]), pk(g[2 * q], g[2 * q + 1]));
        upk(a, acc[2 * q], acc[2 * q + 1]);
    }
#pragma unroll
    for (int c = 0; c < 3; c++) {   // acc_low += SGN * a_mu^dag g
        const float g0r = g[2 * c], g0i = g[2 * c + 1], g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        f2 a2 = pk(acc[12 + 2 * c], acc[12 + 2 * c + 1]), a3 = pk(acc[18 + 2 * c], acc[18 + 2 * c + 1]);
        if (MU == 0) {          // spin 2 += i s g1, spin 3 += i s g0
            a2 = add2(a2, SGN > 0 ? c_i(g1r, g1i) : c_mi(g1r, g1i));
            a3 = add2(a3, SGN > 0 ? c_i(g0r, g0i) : c_mi(g0r, g0i));
        } else if (MU == 1) {   // spin 2 += s g1, spin 3 -= s g0
            a2 = add2(a2, SGN > 0 ? c_pos(g1r, g1i) : c_neg(g1r, g1i));
            a3 = add2(a3, SGN > 0 ? c_neg(g0r, g0i) : c_pos(g0r, g0i));
        } else if (MU == 2) {   // spin 2 += i s g0, spin 3 -= i s g1
            a2 = add2(a2, SGN > 0 ? c_i(g0r, g0i) : c_mi(g0r, g0i));
            a3 = add2(a3, SGN > 0 ? c_mi(g1r, g1i) : c_i(g1r, g1i));
        } else {                // spin 2 += s g0, spin 3 += s g1
            a2 = add2(a2, SGN > 0 ? c_pos(g0r, g0i) : c_neg(g0r, g0i));
            a3 = add2(a3, SGN > 0 ? c_pos(g1r, g1i) : c_neg(g1r, g1i));
        }
        upk(a2, acc[12 + 2 * c], acc[12 + 2 * c + 1]);
        upk(a3, acc[18 + 2 * c], acc[18 + 2 * c + 1]);
    }
}
template <> __device__ __forceinline__ void accumulate<float, 0, 1>(const float* g, float* a) { accumulate_f32<0, 1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 0, -1>(const float* g, float* a) { accumulate_f32<0, -1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 1, 1>(const float* g, float* a) { accumulate_f32<1, 1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 1, -1>(const float* g, float* a) { accumulate_f32<1, -1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 2, 1>(const float* g, float* a) { accumulate_f32<2, 1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 2, -1>(const float* g, float* a) { accumulate_f32<2, -1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 3, 1>(const float* g, float* a) { accumulate_f32<3, 1>(g, a); }
template <> __device__ __forceinline__ void accumulate<float, 3, -1>(const float* g, float* a) { accumulate_f32<3, -1>(g, a); }

// o[c] = sum_c' U[c][c'] h[c'] for fp32: per output colour one FMUL2 and five FFMA2 (U h.re, then (i U) h.im,
// c' = 0, 1, 2).  Non-template overload: chosen over su3_mul<T> for float arguments.
__device__ __forceinline__ void su3_mul(const float* u, const float* h, float* o)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        f2 a = mul2(pk(u[6 * c], u[6 * c + 1]), bc(h[0]));
        a = fma2(c_i(u[6 * c], u[6 * c + 1]), bc(h[1]), a);
        a = fma2(pk(u[6 * c + 2], u[6 * c + 3]), bc(h[2]), a);
        a = fma2(c_i(u[6 * c + 2], u[6 * c + 3]), bc(h[3]), a);
        a = fma2(pk(u[6 * c + 4], u[6 * c + 5]), bc(h[4]), a);
        a = fma2(c_i(u[6 * c + 4], u[6 * c + 5]), bc(h[5]), a);
        upk(a, o[2 * c], o[2 * c + 1]);
    }
}

// z = (cr + i ci) v, z = cr v, z += (cr + i ci) v on arrays of N complex numbers (the epilogue coefficients)
template <int N> __device__ __forceinline__ void cscale_f32(float cr, float ci, const float* v, float* z)
{
#pragma unroll
    for (int q = 0; q < N; q++) {
        const f2 a = fma2(c_i(v[2 * q], v[2 * q + 1]), bc(ci), mul2(pk(v[2 * q], v[2 * q + 1]), bc(cr)));
        upk(a, z[2 * q], z[2 * q + 1]);
    }
}
template <int N> __device__ __forceinline__ void cscale_real_f32(float cr, const float* v, float* z)
{
#pragma unroll
    for (int q = 0; q < N; q++) {
        const f2 a = mul2(pk(v[2 * q], v[2 * q + 1]), bc(cr));
        upk(a, z[2 * q], z[2 * q + 1]);
    }
}
template <int N> __device__ __forceinline__ void caxpy_f32(float cr, float ci, const float* v, float* z)
{
#pragma unroll
    for (int q = 0; q < N; q++) {
        f2 a = fma2(pk(v[2 * q], v[2 * q + 1]), bc(cr), pk(z[2 * q], z[2 * q + 1]));
        a = fma2(c_i(v[2 * q], v[2 * q + 1]), bc(ci), a);
        upk(a, z[2 * q], z[2 * q + 1]);
    }
}

// v *= ph (time-boundary phase on a half spinor), r -= alpha o on N complex numbers
template <int N> __device__ __forceinline__ void rscale_f32(float ph, float* v)
{
#pragma unroll
    for (int q = 0; q < N; q++) {
        const f2 a = mul2(pk(v[2 * q], v[2 * q + 1]), bc(ph));
        upk(a, v[2 * q], v[2 * q + 1]);
    }
}
template <int N> __device__ __forceinline__ void raxpy_f32(float a_, const float* o, float* r)
{
#pragma unroll
    for (int q = 0; q < N; q++) {
        const f2 a = fma2(pk(o[2 * q], o[2 * q + 1]), bc(a_), pk(r[2 * q], r[2 * q + 1]));
        upk(a, r[2 * q], r[2 * q + 1]);
    }
}
