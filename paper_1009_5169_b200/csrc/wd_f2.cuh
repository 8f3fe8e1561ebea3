// wd_f2.cuh -- two lattice sites per thread on Blackwell's packed fp32 pipe (FADD2 / FMUL2 / FFMA2, PTX *.f32x2).
//
// "P32" is the x-paired fp32 form of the native layouts: inside a lattice row of Lx/2 sites of
// one parity, site o < H = Lx/4 (lane A) and site o + H (lane B) share a 128-bit element, one complex number each:
//     float4 = (A.re, B.re, A.im, B.im)
//   spinor row (y, z, t):  [k = 12 complex (spin * 3 + colour)][p = H pairs][r = n columns]   float4
//   link row of (mu, parity): [c = R/2 complex of the row-major 3x3 matrix][p = H]            float4
// so a row is as many bytes as in the plain fp32 form and ONE 128-bit load feeds both lanes of a packed instruction.
// Every hop except +-x maps pair p to pair p with the lanes in place (the two sites are H apart in x and move together);
// a +-x hop that leaves the row's half (p = H-1 -> 0 or 0 -> H-1) lands on the pair with its lanes exchanged.
// Each lane goes through exactly the operations of the scalar kernels (wd_su3.cuh) in the same order, so the results
// are bit for bit theirs.
#pragma once
#include "wd_su3.cuh"

namespace wdp {

struct f2 {
    unsigned long long v;   // lanes (lo = site A, hi = site B), an aligned register pair
};
struct cx2 {
    f2 re, im;
};

__device__ __forceinline__ f2 mk2(float a, float b) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void un2(f2 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v.v)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { f2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return d; }
// ptxas folds the negation into the operand modifier of the consuming FADD2 / FFMA2
__device__ __forceinline__ f2 neg2(f2 a) { float x, y; un2(a, x, y); return mk2(-x, -y); }
__device__ __forceinline__ f2 swap_if(bool c, f2 a) { float x, y; un2(a, x, y); return mk2(c ? y : x, c ? x : y); }
__device__ __forceinline__ f2 zero2() { f2 r; r.v = 0ull; return r; }
// a + S b, a - S b for S = +-1 known at compile time
template <int S> __device__ __forceinline__ f2 addS(f2 a, f2 b) { return S > 0 ? add2(a, b) : sub2(a, b); }
template <int S> __device__ __forceinline__ f2 subS(f2 a, f2 b) { return S > 0 ? sub2(a, b) : add2(a, b); }

// ---- 128-bit element <-> one complex pair --------------------------------------------------------------------
__device__ __forceinline__ cx2 from_vec(const ulonglong2& q) { cx2 c; c.re.v = q.x; c.im.v = q.y; return c; }
__device__ __forceinline__ ulonglong2 to_vec(const cx2& c) { return make_ulonglong2(c.re.v, c.im.v); }

// spinor of pair element e (= p * n + r) of a P32 row; cs = H * n 128-bit elements per complex
__device__ __forceinline__ void ld_spinor(const ulonglong2* __restrict__ row, uint32_t cs, uint32_t e, cx2 (&psi)[12]) {
#pragma unroll
    for (int k = 0; k < 12; ++k) psi[k] = from_vec(row[k * cs + e]);
}
__device__ __forceinline__ void ldg_spinor(const ulonglong2* __restrict__ row, uint32_t cs, uint32_t e, cx2 (&psi)[12]) {
#pragma unroll
    for (int k = 0; k < 12; ++k) psi[k] = from_vec(__ldg(row + k * cs + e));
}
__device__ __forceinline__ void st_spinor(ulonglong2* __restrict__ row, uint32_t cs, uint32_t e, const cx2 (&psi)[12]) {
#pragma unroll
    for (int k = 0; k < 12; ++k) row[k * cs + e] = to_vec(psi[k]);
}
// link of pair p of a P32 link row; H pairs per complex: the RECON / 2 stored complex numbers
template <int RECON>
__device__ __forceinline__ void ld_link_raw(const ulonglong2* __restrict__ row, uint32_t H, uint32_t p, cx2 (&u)[9]) {
#pragma unroll
    for (int c = 0; c < RECON / 2; ++c) u[c] = from_vec(row[c * H + p]);
}
// RECON == 12: row 3 rebuilt as in wd_su3.cuh rebuild_row3
template <int RECON>
__device__ __forceinline__ void finish_link(cx2 (&u)[9]) {
    if (RECON == 12) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int a = (k + 1) % 3, b = (k + 2) % 3;
            f2 re = mul2(u[a].re, u[3 + b].re);
            re = fma2(neg2(u[a].im), u[3 + b].im, re);
            re = fma2(neg2(u[b].re), u[3 + a].re, re);
            re = fma2(u[b].im, u[3 + a].im, re);
            f2 im = mul2(u[b].re, u[3 + a].im);
            im = fma2(u[b].im, u[3 + a].re, im);
            im = fma2(neg2(u[a].re), u[3 + b].im, im);
            im = fma2(neg2(u[a].im), u[3 + b].re, im);
            u[6 + k].re = re;
            u[6 + k].im = im;
        }
    }
}
template <int RECON>
__device__ __forceinline__ void ld_link(const ulonglong2* __restrict__ row, uint32_t H, uint32_t p, cx2 (&u)[9]) {
    ld_link_raw<RECON>(row, H, p, u);
    finish_link<RECON>(u);
}

// ---- spin projection (1 - SIGMA gamma_MU) psi -> hs[0..2] = h0, hs[3..5] = h1 (wd_su3.cuh project, per lane) ----
template <int MU, int SIGMA>
__device__ __forceinline__ void project(const cx2 (&psi)[12], cx2 (&hs)[6]) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const cx2 u0 = psi[a], u1 = psi[3 + a], l0 = psi[6 + a], l1 = psi[9 + a];
        if (MU == 0) {
            hs[a].re = subS<SIGMA>(u0.re, l1.im);     hs[a].im = addS<SIGMA>(u0.im, l1.re);
            hs[3 + a].re = subS<SIGMA>(u1.re, l0.im); hs[3 + a].im = addS<SIGMA>(u1.im, l0.re);
        } else if (MU == 1) {
            hs[a].re = addS<SIGMA>(u0.re, l1.re);     hs[a].im = addS<SIGMA>(u0.im, l1.im);
            hs[3 + a].re = subS<SIGMA>(u1.re, l0.re); hs[3 + a].im = subS<SIGMA>(u1.im, l0.im);
        } else if (MU == 2) {
            hs[a].re = subS<SIGMA>(u0.re, l0.im);     hs[a].im = addS<SIGMA>(u0.im, l0.re);
            hs[3 + a].re = addS<SIGMA>(u1.re, l1.im); hs[3 + a].im = subS<SIGMA>(u1.im, l1.re);
        } else {
            hs[a].re = subS<SIGMA>(u0.re, l0.re);     hs[a].im = subS<SIGMA>(u0.im, l0.im);
            hs[3 + a].re = subS<SIGMA>(u1.re, l1.re); hs[3 + a].im = subS<SIGMA>(u1.im, l1.im);
        }
    }
}

// ---- acc += reconstruct(chi) (wd_su3.cuh accumulate, per lane); FIRST: acc is taken as zero ---------------------
template <int S, bool FIRST> __device__ __forceinline__ f2 accP(f2 acc, f2 c) {   // acc + S c
    if (FIRST) return S > 0 ? c : neg2(c);
    return S > 0 ? add2(acc, c) : sub2(acc, c);
}
template <int MU, int SIGMA, bool FIRST>
__device__ __forceinline__ void accumulate(cx2 (&acc)[12], const cx2 (&chi)[6]) {
    constexpr int P = SIGMA, M = -SIGMA;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const cx2 c0 = chi[a], c1 = chi[3 + a];
        acc[a].re = accP<1, FIRST>(acc[a].re, c0.re);         acc[a].im = accP<1, FIRST>(acc[a].im, c0.im);
        acc[3 + a].re = accP<1, FIRST>(acc[3 + a].re, c1.re); acc[3 + a].im = accP<1, FIRST>(acc[3 + a].im, c1.im);
        if (MU == 0) {         // lower = (-s i c1, -s i c0)
            acc[6 + a].re = accP<P, FIRST>(acc[6 + a].re, c1.im); acc[6 + a].im = accP<M, FIRST>(acc[6 + a].im, c1.re);
            acc[9 + a].re = accP<P, FIRST>(acc[9 + a].re, c0.im); acc[9 + a].im = accP<M, FIRST>(acc[9 + a].im, c0.re);
        } else if (MU == 1) {  // lower = (-s c1, +s c0)
            acc[6 + a].re = accP<M, FIRST>(acc[6 + a].re, c1.re); acc[6 + a].im = accP<M, FIRST>(acc[6 + a].im, c1.im);
            acc[9 + a].re = accP<P, FIRST>(acc[9 + a].re, c0.re); acc[9 + a].im = accP<P, FIRST>(acc[9 + a].im, c0.im);
        } else if (MU == 2) {  // lower = (-s i c0, +s i c1)
            acc[6 + a].re = accP<P, FIRST>(acc[6 + a].re, c0.im); acc[6 + a].im = accP<M, FIRST>(acc[6 + a].im, c0.re);
            acc[9 + a].re = accP<M, FIRST>(acc[9 + a].re, c1.im); acc[9 + a].im = accP<P, FIRST>(acc[9 + a].im, c1.re);
        } else {               // lower = (-s c0, -s c1)
            acc[6 + a].re = accP<M, FIRST>(acc[6 + a].re, c0.re); acc[6 + a].im = accP<M, FIRST>(acc[6 + a].im, c0.im);
            acc[9 + a].re = accP<M, FIRST>(acc[9 + a].re, c1.re); acc[9 + a].im = accP<M, FIRST>(acc[9 + a].im, c1.im);
        }
    }
}

// chi_j = U h_j (ADJ = false) or U^dag h_j (ADJ = true): 12 FMUL2 + 60 FFMA2 for two sites (wd_su3.cuh su3_mul)
template <bool ADJ>
__device__ __forceinline__ void su3_mul(const cx2 (&u)[9], const cx2 (&hs)[6], cx2 (&chi)[6]) {
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            f2 re, im;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const cx2 m = ADJ ? u[c * 3 + a] : u[a * 3 + c];
                const cx2 v = hs[3 * j + c];
                if (c == 0) { re = mul2(m.re, v.re); im = mul2(m.re, v.im); }
                else        { re = fma2(m.re, v.re, re); im = fma2(m.re, v.im, im); }
                if (ADJ) {
                    re = fma2(m.im, v.im, re);
                    im = fma2(neg2(m.im), v.re, im);
                } else {
                    re = fma2(neg2(m.im), v.im, re);
                    im = fma2(m.im, v.re, im);
                }
            }
            chi[3 * j + a].re = re;
            chi[3 * j + a].im = im;
        }
}

}  // namespace wdp
