// wd_su3.cuh -- register-level building blocks shared by the hop and force kernels: complex type,
// 128-bit spinor/link loads from the native layouts, 12-real link rebuild, half-spinor projection
// (DESIGN.md section 6a "Half-spinor projection"; chiral gamma basis), SU(3) x colour-vector product.
#pragma once
#include "wd_internal.h"

namespace wdk {

template <typename T>
struct cx {
    T re, im;
};

template <typename T> struct Vec;
template <> struct Vec<float> { typedef float4 type; enum { NCH = 6 }; };
template <> struct Vec<double> { typedef double2 type; enum { NCH = 12 }; };

// ---- loads / stores of one spinor (12 complex) at vec index `e` of a half-lattice block ----------
template <typename I>
__device__ __forceinline__ void load_spinor(const float4* __restrict__ base, I stride, I e, cx<float> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float4 v = __ldg(base + c * stride + e);
        psi[2 * c].re = v.x; psi[2 * c].im = v.y; psi[2 * c + 1].re = v.z; psi[2 * c + 1].im = v.w;
    }
}
template <typename I>
__device__ __forceinline__ void load_spinor(const double2* __restrict__ base, I stride, I e, cx<double> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        const double2 v = __ldg(base + c * stride + e);
        psi[c].re = v.x; psi[c].im = v.y;
    }
}
template <typename I>
__device__ __forceinline__ void store_spinor(float4* __restrict__ base, I stride, I e, const cx<float> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 6; ++c)
        base[c * stride + e] = make_float4(psi[2 * c].re, psi[2 * c].im, psi[2 * c + 1].re, psi[2 * c + 1].im);
}
template <typename I>
__device__ __forceinline__ void store_spinor(double2* __restrict__ base, I stride, I e, const cx<double> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 12; ++c) base[c * stride + e] = make_double2(psi[c].re, psi[c].im);
}

// ---- link load: 9 complex, row-major; RECON==12 rebuilds row 3 = conj(row1 x row2) ----------------
template <int RECON, typename I>
__device__ __forceinline__ void load_link(const float* __restrict__ blk, I Vh, I h, cx<float> (&u)[9]) {
    const float4* q = reinterpret_cast<const float4*>(blk);
#pragma unroll
    for (int c = 0; c < (RECON == 18 ? 4 : 3); ++c) {
        const float4 v = __ldg(q + c * Vh + h);
        u[2 * c].re = v.x; u[2 * c].im = v.y; u[2 * c + 1].re = v.z; u[2 * c + 1].im = v.w;
    }
    if (RECON == 18) {
        const float2 w = __ldg(reinterpret_cast<const float2*>(blk) + (8 * Vh + h));
        u[8].re = w.x; u[8].im = w.y;
    }
}
template <int RECON, typename I>
__device__ __forceinline__ void load_link(const double* __restrict__ blk, I Vh, I h, cx<double> (&u)[9]) {
    const double2* q = reinterpret_cast<const double2*>(blk);
#pragma unroll
    for (int c = 0; c < (RECON == 18 ? 9 : 6); ++c) {
        const double2 v = __ldg(q + c * Vh + h);
        u[c].re = v.x; u[c].im = v.y;
    }
}
template <typename T>
__device__ __forceinline__ void rebuild_row3(cx<T> (&u)[9]) {
    // u[6+k] = conj( u[(k+1)%3] * u[3+(k+2)%3] - u[(k+2)%3] * u[3+(k+1)%3] ), as explicit FMA chains
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int a = (k + 1) % 3, b = (k + 2) % 3;
        T re = u[a].re * u[3 + b].re;
        re = fma(-u[a].im, u[3 + b].im, re);
        re = fma(-u[b].re, u[3 + a].re, re);
        re = fma(u[b].im, u[3 + a].im, re);
        T im = u[b].re * u[3 + a].im;          // this is -Im(...)
        im = fma(u[b].im, u[3 + a].re, im);
        im = fma(-u[a].re, u[3 + b].im, im);
        im = fma(-u[a].im, u[3 + b].re, im);
        u[6 + k].re = re;
        u[6 + k].im = im;
    }
}

// ---- spin projection (1 - SIGMA gamma_MU) psi -> half spinor hs[0..2] = h0, hs[3..5] = h1 ---------
template <int MU, int SIGMA, typename T>
__device__ __forceinline__ void project(const cx<T> (&psi)[12], cx<T> (&hs)[6]) {
    const T s = (T)SIGMA;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const cx<T> u0 = psi[a], u1 = psi[3 + a], l0 = psi[6 + a], l1 = psi[9 + a];
        if (MU == 0) {         // h0 = u0 + s i l1 ; h1 = u1 + s i l0
            hs[a].re = u0.re - s * l1.im;     hs[a].im = u0.im + s * l1.re;
            hs[3 + a].re = u1.re - s * l0.im; hs[3 + a].im = u1.im + s * l0.re;
        } else if (MU == 1) {  // h0 = u0 + s l1 ; h1 = u1 - s l0
            hs[a].re = u0.re + s * l1.re;     hs[a].im = u0.im + s * l1.im;
            hs[3 + a].re = u1.re - s * l0.re; hs[3 + a].im = u1.im - s * l0.im;
        } else if (MU == 2) {  // h0 = u0 + s i l0 ; h1 = u1 - s i l1
            hs[a].re = u0.re - s * l0.im;     hs[a].im = u0.im + s * l0.re;
            hs[3 + a].re = u1.re + s * l1.im; hs[3 + a].im = u1.im - s * l1.re;
        } else {               // h0 = u0 - s l0 ; h1 = u1 - s l1
            hs[a].re = u0.re - s * l0.re;     hs[a].im = u0.im - s * l0.im;
            hs[3 + a].re = u1.re - s * l1.re; hs[3 + a].im = u1.im - s * l1.im;
        }
    }
}

// ---- acc += reconstruct(chi): upper = (chi0, chi1), lower from the same table ---------------------
// FIRST: acc is taken as zero (the first of the eight directions), which saves the 24 additions to 0.
template <int MU, int SIGMA, bool FIRST = false, typename T>
__device__ __forceinline__ void accumulate(cx<T> (&acc)[12], const cx<T> (&chi)[6]) {
    const T s = (T)SIGMA;
    if (FIRST) {
#pragma unroll
        for (int k = 0; k < 12; ++k) { acc[k].re = 0; acc[k].im = 0; }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const cx<T> c0 = chi[a], c1 = chi[3 + a];
        acc[a].re += c0.re;     acc[a].im += c0.im;
        acc[3 + a].re += c1.re; acc[3 + a].im += c1.im;
        if (MU == 0) {         // lower = (-s i c1, -s i c0)
            acc[6 + a].re += s * c1.im; acc[6 + a].im -= s * c1.re;
            acc[9 + a].re += s * c0.im; acc[9 + a].im -= s * c0.re;
        } else if (MU == 1) {  // lower = (-s c1, +s c0)
            acc[6 + a].re -= s * c1.re; acc[6 + a].im -= s * c1.im;
            acc[9 + a].re += s * c0.re; acc[9 + a].im += s * c0.im;
        } else if (MU == 2) {  // lower = (-s i c0, +s i c1)
            acc[6 + a].re += s * c0.im; acc[6 + a].im -= s * c0.re;
            acc[9 + a].re -= s * c1.im; acc[9 + a].im += s * c1.re;
        } else {               // lower = (-s c0, -s c1)
            acc[6 + a].re -= s * c0.re; acc[6 + a].im -= s * c0.im;
            acc[9 + a].re -= s * c1.re; acc[9 + a].im -= s * c1.im;
        }
    }
}

// chi_j = U h_j (ADJ = false) or U^dag h_j (ADJ = true), j = 0, 1.  Written as explicit FMA chains:
// 12 FMUL + 60 FFMA per call (the compiler may not re-associate `re += a*b - c*d` into two FMAs).
template <bool ADJ, typename T>
__device__ __forceinline__ void su3_mul(const cx<T> (&u)[9], const cx<T> (&hs)[6], cx<T> (&chi)[6]) {
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            T re, im;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const cx<T> m = ADJ ? u[c * 3 + a] : u[a * 3 + c];
                const cx<T> v = hs[3 * j + c];
                if (c == 0) { re = m.re * v.re; im = m.re * v.im; }
                else        { re = fma(m.re, v.re, re); im = fma(m.re, v.im, im); }
                if (ADJ) {  // conj(m) * v
                    re = fma(m.im, v.im, re);
                    im = fma(-m.im, v.re, im);
                } else {
                    re = fma(-m.im, v.im, re);
                    im = fma(m.im, v.re, im);
                }
            }
            chi[3 * j + a].re = re;
            chi[3 * j + a].im = im;
        }
}

}  // namespace wdk
