// wd_h16.cuh -- 16-bit storage of spinor blocks for the inner solver ("we follow the tuning
// techniques described in [4]": half-precision storage with single-precision arithmetic).
//
// Format "H16" of a HALF-lattice block of n columns, row-major layout blocks as the fp32 native form (block b = one
// lattice row of RB = Lx/2 sites; requires RB * n to be a multiple of 4):
//     block b:  uint4 [k = 3][o = RB][n]     8 halves each: reals 8k .. 8k+7 of the 24 reals (spin, colour, re/im) of a spinor
//               float [o = RB][n]            scale = max |real| of that spinor
//   value = scale * half;  52 bytes per site and column instead of 96, 13 RB n / 4 16-byte units per block.
// Arithmetic is always fp32: these helpers convert on load and store.  The per-spinor scale keeps the relative precision
// of 2^-11 whatever the magnitude of the vector (the residual falls by twelve orders of magnitude during a solve).
#pragma once
#include <cuda_fp16.h>

#include "wd_su3.cuh"

namespace wdh {

// 16-byte units of one layout block (row) of an H16 half-lattice block with rbn = RB * n
__host__ __device__ __forceinline__ uint32_t h16_row_vecs(uint32_t rbn) { return 13 * rbn / 4; }

template <bool SCALE = true>
__device__ __forceinline__ void h16_expand(const float4& q, float s, wdk::cx<float>* out) {
    const __half2* h = reinterpret_cast<const __half2*>(&q);
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const float2 f = __half22float2(h[m]);
        out[m].re = SCALE ? s * f.x : f.x;
        out[m].im = SCALE ? s * f.y : f.y;
    }
}

// spinor (site, column) element e of the row at `row` (16-byte units); rbn = RB * n.  LDG: through the read-only path.
template <bool LDG>
__device__ __forceinline__ void h16_load(const float4* __restrict__ row, uint32_t rbn, uint32_t e, wdk::cx<float> (&psi)[12]) {
    float4 q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) q[k] = LDG ? __ldg(row + k * rbn + e) : row[k * rbn + e];
    const float* sp = reinterpret_cast<const float*>(row + 3 * rbn) + e;
    const float s = LDG ? __ldg(sp) : *sp;
#pragma unroll
    for (int k = 0; k < 3; ++k) h16_expand(q[k], s, &psi[4 * k]);
}

// the same without applying the scale (the hop applies it to the 12 reals AFTER spin projection and the SU(3) product,
// which are linear: 12 multiplications per neighbour instead of 24)
__device__ __forceinline__ float h16_load_raw(const float4* __restrict__ row, uint32_t rbn, uint32_t e, wdk::cx<float> (&psi)[12]) {
    float4 q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) q[k] = row[k * rbn + e];
    const float s = reinterpret_cast<const float*>(row + 3 * rbn)[e];
#pragma unroll
    for (int k = 0; k < 3; ++k) h16_expand<false>(q[k], 1.f, &psi[4 * k]);
    return s;
}

__device__ __forceinline__ void h16_store(float4* __restrict__ row, uint32_t rbn, uint32_t e, const wdk::cx<float> (&psi)[12]) {
    float m = 0.f;
#pragma unroll
    for (int k = 0; k < 12; ++k) m = fmaxf(m, fmaxf(fabsf(psi[k].re), fabsf(psi[k].im)));
    const float inv = m > 0.f ? 1.f / m : 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        float4 q;
        __half2* h = reinterpret_cast<__half2*>(&q);
#pragma unroll
        for (int j = 0; j < 4; ++j) h[j] = __floats2half2_rn(psi[4 * k + j].re * inv, psi[4 * k + j].im * inv);
        row[k * rbn + e] = q;
    }
    reinterpret_cast<float*>(row + 3 * rbn)[e] = m;
}

}  // namespace wdh
