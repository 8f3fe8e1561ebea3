// wd_layout.cu -- canonical <-> native conversions (hot-path step a0 "gauge ingest" and the
// pack/unpack of spinor blocks).  Conversion only: no arithmetic of the method happens here.
//
// Native storage cuts the V/2 sites of a parity into layout blocks of RB consecutive sites (wd_internal.h:
// RB = Lx/2, one lattice row, in the linear site order; RB = V/2 in the tiled order); site h = b*RB + o.
// Links, per precision and link form (R = 18 or 12 reals): the array of (mu, parity) starts at real offset
//   (mu*2+parity)*R*Vh; layout block b starts R*RB*b reals further and holds
//   fp64: double2 chunk c (= complex c of the row-major 3x3 matrix, rows 1-2 only for R=12) at double2 index
//         c*RB + o;
//   fp32: float4 chunk c (= complex 2c, 2c+1) at float offset c*4*RB + 4*o, c < R/4; for R=18 the ninth
//         complex is a float2 at float offset 16*RB + 2*o.
// Spinor blocks: element (parity p, chunk k, site h, column r) at 128-bit index
//   p*NCH*Vh*n + ((b*NCH + k)*RB + o)*n + r,   NCH = 12 (fp64, one complex) or 6 (fp32, complex 2k and 2k+1).
#include "wd_internal.h"

namespace {

__global__ void gauge_ingest_kernel(const double* __restrict__ U, const int32_t* __restrict__ site_of, long V,
                                    long Vh, long RB, double* __restrict__ u64_18, double* __restrict__ u64_12,
                                    float* __restrict__ u32_18, float* __restrict__ u32_12,
                                    float* __restrict__ p32_18, float* __restrict__ p32_12) {
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 4 * 2 * Vh) return;
    const long h = tid % Vh;
    const int p = (int)((tid / Vh) & 1);
    const int mu = (int)(tid / (2 * Vh));
    const long s = site_of[p * Vh + h];
    const double* u = U + ((long)mu * V + s) * 18;
    double v[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) v[k] = u[k];
    const long blk = (long)(mu * 2 + p);
    const long lb = h / RB, o = h - lb * RB;  // layout block and offset inside it
    double* a = u64_18 + blk * 18 * Vh + lb * 18 * RB;
    double* b = u64_12 + blk * 12 * Vh + lb * 12 * RB;
#pragma unroll
    for (int c = 0; c < 9; ++c) {
        a[(c * RB + o) * 2] = v[2 * c];
        a[(c * RB + o) * 2 + 1] = v[2 * c + 1];
        if (c < 6) {
            b[(c * RB + o) * 2] = v[2 * c];
            b[(c * RB + o) * 2 + 1] = v[2 * c + 1];
        }
    }
    float* fa = u32_18 + blk * 18 * Vh + lb * 18 * RB;
    float* fb = u32_12 + blk * 12 * Vh + lb * 12 * RB;
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            fa[c * 4 * RB + 4 * o + j] = (float)v[4 * c + j];
            if (c < 3) fb[c * 4 * RB + 4 * o + j] = (float)v[4 * c + j];
        }
    fa[16 * RB + 2 * o] = (float)v[16];
    fa[16 * RB + 2 * o + 1] = (float)v[17];
    if (p32_18) {   // P32 (wd_f2.cuh): float4 (A.re, B.re, A.im, B.im) of complex c at index c * H + pair, H = RB / 2
        const long H = RB / 2, pr = o % H, lane = o / H;
        float* pa = p32_18 + blk * 18 * Vh + lb * 18 * RB;
        float* pb = p32_12 + blk * 12 * Vh + lb * 12 * RB;
#pragma unroll
        for (int c = 0; c < 9; ++c) {
            pa[(c * H + pr) * 4 + lane] = (float)v[2 * c];
            pa[(c * H + pr) * 4 + 2 + lane] = (float)v[2 * c + 1];
            if (c < 6) {
                pb[(c * H + pr) * 4 + lane] = (float)v[2 * c];
                pb[(c * H + pr) * 4 + 2 + lane] = (float)v[2 * c + 1];
            }
        }
    }
}

template <typename T, bool PAIRED = false>
__global__ void pack_kernel(const double* __restrict__ canon, const int32_t* __restrict__ site_of,
                            const int32_t* __restrict__ nbr, long V, long Vh, long RB, int n, T* __restrict__ native) {
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * Vh * n) return;
    const int r = (int)(tid % n);
    const long ph = tid / n;
    const long h = ph % Vh;
    const int p = (int)(ph / Vh);
    const long lb = h / RB, o = h - lb * RB;
    const long s = site_of[ph];
    const bool frozen = ((uint32_t)nbr[ph * WD_NDIR] & WD_SITE_FROZEN) != 0;
    const double* src = canon + ((long)r * V + s) * 24;
    double v[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) v[k] = frozen ? 0.0 : src[k];
    if (sizeof(T) == 8) {
        double* dst = (double*)native;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const long e = ((long)p * 12 * Vh * n + ((lb * 12 + k) * RB + o) * n + r) * 2;
            dst[e] = v[2 * k];
            dst[e + 1] = v[2 * k + 1];
        }
    } else if (PAIRED) {   // P32: complex k of pair (o % H) at element ((lb*12 + k)*H + pair)*n + r, lane o / H
        float* dst = (float*)native;
        const long H = RB / 2, pr = o % H, lane = o / H;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const long e = ((long)p * 6 * Vh * n + ((lb * 12 + k) * H + pr) * n + r) * 4;
            dst[e + lane] = (float)v[2 * k];
            dst[e + 2 + lane] = (float)v[2 * k + 1];
        }
    } else {
        float* dst = (float*)native;
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            const long e = ((long)p * 6 * Vh * n + ((lb * 6 + c) * RB + o) * n + r) * 4;
#pragma unroll
            for (int j = 0; j < 4; ++j) dst[e + j] = (float)v[4 * c + j];
        }
    }
}

template <typename T, bool PAIRED = false>
__global__ void unpack_kernel(const T* __restrict__ native, const int32_t* __restrict__ site_of, long V, long Vh,
                              long RB, int n, double* __restrict__ canon) {
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * Vh * n) return;
    const int r = (int)(tid % n);
    const long ph = tid / n;
    const long h = ph % Vh;
    const int p = (int)(ph / Vh);
    const long lb = h / RB, o = h - lb * RB;
    const long s = site_of[ph];
    double* dst = canon + ((long)r * V + s) * 24;
    if (sizeof(T) == 8) {
        const double* src = (const double*)native;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const long e = ((long)p * 12 * Vh * n + ((lb * 12 + k) * RB + o) * n + r) * 2;
            dst[2 * k] = src[e];
            dst[2 * k + 1] = src[e + 1];
        }
    } else if (PAIRED) {
        const float* src = (const float*)native;
        const long H = RB / 2, pr = o % H, lane = o / H;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const long e = ((long)p * 6 * Vh * n + ((lb * 12 + k) * H + pr) * n + r) * 4;
            dst[2 * k] = (double)src[e + lane];
            dst[2 * k + 1] = (double)src[e + 2 + lane];
        }
    } else {
        const float* src = (const float*)native;
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            const long e = ((long)p * 6 * Vh * n + ((lb * 6 + c) * RB + o) * n + r) * 4;
#pragma unroll
            for (int j = 0; j < 4; ++j) dst[4 * c + j] = (double)src[e + j];
        }
    }
}

}  // namespace

int wd_layout_gauge(wd_ctx* c, const double* U) {
    const long total = 8 * c->Vh;
    const int B = 128;
    wd_prof_scope prof(c, WD_PROF_LAYOUT);
    gauge_ingest_kernel<<<(unsigned)((total + B - 1) / B), B, 0, c->stream>>>(
        U, c->d_site_of, c->V, c->Vh, (long)c->RB, c->d_U64[0], c->d_U64[1], c->d_U32[0], c->d_U32[1], c->d_U32P[0], c->d_U32P[1]);
    WD_LAUNCH_CHECK(c);
    return WD_OK;
}

int wd_layout_pack(wd_ctx* c, int prec, int n, const double* canon, void* native) {
    const long total = 2 * c->Vh * n;
    const int B = 128;
    const unsigned G = (unsigned)((total + B - 1) / B);
    wd_prof_scope prof(c, WD_PROF_LAYOUT);
    if (prec == WD_F64)
        pack_kernel<double><<<G, B, 0, c->stream>>>(canon, c->d_site_of, c->d_nbr, c->V, c->Vh, (long)c->RB, n, (double*)native);
    else if (prec == WD_F32P)
        pack_kernel<float, true><<<G, B, 0, c->stream>>>(canon, c->d_site_of, c->d_nbr, c->V, c->Vh, (long)c->RB, n, (float*)native);
    else
        pack_kernel<float><<<G, B, 0, c->stream>>>(canon, c->d_site_of, c->d_nbr, c->V, c->Vh, (long)c->RB, n, (float*)native);
    WD_LAUNCH_CHECK(c);
    return WD_OK;
}

int wd_layout_unpack(wd_ctx* c, int prec, int n, const void* native, double* canon) {
    const long total = 2 * c->Vh * n;
    const int B = 128;
    const unsigned G = (unsigned)((total + B - 1) / B);
    wd_prof_scope prof(c, WD_PROF_LAYOUT);
    if (prec == WD_F64)
        unpack_kernel<double><<<G, B, 0, c->stream>>>((const double*)native, c->d_site_of, c->V, c->Vh, (long)c->RB, n, canon);
    else if (prec == WD_F32P)
        unpack_kernel<float, true><<<G, B, 0, c->stream>>>((const float*)native, c->d_site_of, c->V, c->Vh, (long)c->RB, n, canon);
    else
        unpack_kernel<float><<<G, B, 0, c->stream>>>((const float*)native, c->d_site_of, c->V, c->Vh, (long)c->RB, n, canon);
    WD_LAUNCH_CHECK(c);
    return WD_OK;
}
