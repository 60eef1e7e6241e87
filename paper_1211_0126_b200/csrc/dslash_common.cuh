// dslash_common.cuh -- spin projection / reconstruction shared by the stencil kernels (H5).
// gamma_mu = [[0, a_mu], [a_mu^dag, 0]] in the chiral basis C3: (1 +- gamma_mu) psi = [h; +- a_mu^dag h]
// with h = psi_up +- a_mu psi_low, so the SU(3) multiply acts on 2 spin x 3 colour only.
#pragma once
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
        for (int j = 0; j < 4; j++) {
            float p = v[6 * j] * v[6 * j];
#pragma unroll
            for (int k = 1; k < 6; k++) p = fmaf(v[6 * j + k], v[6 * j + k], p);
            s += (double)p;
        }
    }
    return s;
}
