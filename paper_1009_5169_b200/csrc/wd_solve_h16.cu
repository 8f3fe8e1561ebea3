// wd_solve_h16.cu -- the lower-traffic inner solver ("tuning techniques described in [4]"):
// BiCGStab whose vectors are STORED in 16 bits (wd_h16.cuh: fp16 mantissas + one fp32 scale per spinor), computed in
// fp32, kept honest by RELIABLE UPDATES instead of restarts.
//
//   even/odd system  Ahat X_e = Bhat  (as wd_solve.cu);  Y (fp64) = 0, x (fp32) = 0, r = r~ = Bhat_i / |Bhat_i|  (H16)
//   one continuous BiCGStab sequence per column (textbook recurrence) on r, p, v, s, t in H16,
//   x accumulated in fp32.  When a column's recursive |r| has fallen below delta times its largest value since the last
//   update (or every column looks converged), a reliable update:
//        Y += |Bhat_i| x ; x = 0 ;  R = Bhat - Ahat Y  in fp64 (the TRUE residual) ;  stop if |R_i| <= tol |phi_i| for all i ;
//        r = R_i / |Bhat_i|  (H16) ;  rho = <r~, r>, beta recomputed with the rho of the previous iteration ;  go on with the
//        same p, v, alpha, omega: the Krylov space is kept, which a defect-correction restart throws away.
//   Half the bytes per vector pass (52 instead of 96 per site and column) in the BLAS1 kernels and in the hop's spinor
//   operands; the links stay fp32.  Served by the z-march hop kernel only (row-major layout, n_rhs >= 3, Lx/2 * n_rhs a
//   multiple of 4); wd_solve_impl falls back to the fp32-storage solver elsewhere.
#include <chrono>

#include "wd_blas.cuh"
#include "wd_h16.cuh"

using namespace wdblas;
using namespace wdh;
using wdk::cx;

namespace {

struct Geo {
    long items;      // Vh * n
    uint32_t RB, n, rbn, rowH;   // rowH = 16-byte units of an H16 row
};

#define WD_H16_PROLOGUE                                                                 \
    const int r = threadIdx.x % G.n;                                                    \
    const long stride = (long)gridDim.x * blockDim.x;                                   \
    const long i0 = (long)blockIdx.x * blockDim.x + threadIdx.x;                        \
    const long cnt = i0 < G.items ? (G.items - 1 - i0) / stride + 1 : 0;

// item i = h * n + r  ->  (layout block b, element e inside a chunk of the block)
__device__ __forceinline__ void locate(const Geo& G, long i, uint32_t* b, uint32_t* e) {
    const uint32_t h = (uint32_t)(i / G.n);
    const uint32_t o = h % G.RB;
    *b = h / G.RB;
    *e = o * G.n + (uint32_t)(i % G.n);
}

__device__ __forceinline__ void load32(const float4* __restrict__ X, const Geo& G, uint32_t b, uint32_t e, cx<float> (&x)[12]) {
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float4 v = X[(size_t)(b * 6 + c) * G.rbn + e];
        x[2 * c].re = v.x; x[2 * c].im = v.y; x[2 * c + 1].re = v.z; x[2 * c + 1].im = v.w;
    }
}
__device__ __forceinline__ void store32(float4* __restrict__ X, const Geo& G, uint32_t b, uint32_t e, const cx<float> (&x)[12]) {
#pragma unroll
    for (int c = 0; c < 6; ++c) X[(size_t)(b * 6 + c) * G.rbn + e] = make_float4(x[2 * c].re, x[2 * c].im, x[2 * c + 1].re, x[2 * c + 1].im);
}

// P = R + beta (P - omega V)
__global__ void h16_p_update(Geo G, int rev, const double* __restrict__ scal, const float4* __restrict__ R, float4* __restrict__ P,
                             const float4* __restrict__ V) {
    if (scal[G_DONE] != 0.0) return;
    WD_H16_PROLOGUE
    const float br = (float)scal[S_BETA_RE * WD_MAX_RHS + r], bi = (float)scal[S_BETA_IM * WD_MAX_RHS + r];
    const float wr = (float)scal[S_OMEGA_RE * WD_MAX_RHS + r], wi = (float)scal[S_OMEGA_IM * WD_MAX_RHS + r];
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;
        uint32_t b, e;
        locate(G, i, &b, &e);
        cx<float> a[12], p[12], v[12];
        h16_load<false>(R + (size_t)b * G.rowH, G.rbn, e, a);
        h16_load<false>(P + (size_t)b * G.rowH, G.rbn, e, p);
        h16_load<false>(V + (size_t)b * G.rowH, G.rbn, e, v);
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            const float tr = p[c].re - (wr * v[c].re - wi * v[c].im);
            const float ti = p[c].im - (wr * v[c].im + wi * v[c].re);
            p[c].re = a[c].re + (br * tr - bi * ti);
            p[c].im = a[c].im + (br * ti + bi * tr);
        }
        h16_store(P + (size_t)b * G.rowH, G.rbn, e, p);
    }
}

// S = R - alpha V   (in place on R)
__global__ void h16_s_update(Geo G, int rev, const double* __restrict__ scal, float4* __restrict__ R, const float4* __restrict__ V) {
    if (scal[G_DONE] != 0.0) return;
    WD_H16_PROLOGUE
    const float ar = (float)scal[S_ALPHA_RE * WD_MAX_RHS + r], ai = (float)scal[S_ALPHA_IM * WD_MAX_RHS + r];
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;
        uint32_t b, e;
        locate(G, i, &b, &e);
        cx<float> a[12], v[12];
        h16_load<false>(R + (size_t)b * G.rowH, G.rbn, e, a);
        h16_load<false>(V + (size_t)b * G.rowH, G.rbn, e, v);
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            a[c].re -= ar * v[c].re - ai * v[c].im;
            a[c].im -= ar * v[c].im + ai * v[c].re;
        }
        h16_store(R + (size_t)b * G.rowH, G.rbn, e, a);
    }
}

// X (fp32) += alpha P + omega S;  R = S - omega T;  <Rt, R>, |R|^2  ->  rho, beta, convergence / reliable-update flags.
// Worked chunk by chunk (8 reals of every operand at a time) so that only the new r (24 reals) lives across the loop:
// ~80 registers instead of ~150 with all five operands expanded at once.
__global__ void __launch_bounds__(512) h16_xr_update(Geo G, int rev, RedBuf rb, float4* __restrict__ X, const float4* __restrict__ P,
                                                     float4* __restrict__ R, const float4* __restrict__ Tt, const float4* __restrict__ Rt) {
    if (rb.scal[G_DONE] != 0.0) return;
    WD_H16_PROLOGUE
    const double* scal = rb.scal;
    const float ar = (float)scal[S_ALPHA_RE * WD_MAX_RHS + r], ai = (float)scal[S_ALPHA_IM * WD_MAX_RHS + r];
    const float wr = (float)scal[S_OMEGA_RE * WD_MAX_RHS + r], wi = (float)scal[S_OMEGA_IM * WD_MAX_RHS + r];
    double s[3] = {0.0, 0.0, 0.0};
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;
        uint32_t b, e;
        locate(G, i, &b, &e);
        const float4* Pr = P + (size_t)b * G.rowH;
        float4* Rr = R + (size_t)b * G.rowH;
        const float4* Tr = Tt + (size_t)b * G.rowH;
        const float4* Qr = Rt + (size_t)b * G.rowH;
        const float sp = reinterpret_cast<const float*>(Pr + 3 * G.rbn)[e], ss = reinterpret_cast<const float*>(Rr + 3 * G.rbn)[e];
        const float st = reinterpret_cast<const float*>(Tr + 3 * G.rbn)[e], sq = reinterpret_cast<const float*>(Qr + 3 * G.rbn)[e];
        cx<float> rn[12];
        float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            cx<float> p[4], sv[4], t[4], q[4];
            h16_expand(Pr[c * G.rbn + e], sp, p);
            h16_expand(Rr[c * G.rbn + e], ss, sv);
            h16_expand(Tr[c * G.rbn + e], st, t);
            h16_expand(Qr[c * G.rbn + e], sq, q);
            float4 xa = X[(size_t)(b * 6 + 2 * c) * G.rbn + e], xb = X[(size_t)(b * 6 + 2 * c + 1) * G.rbn + e];
            float* xv[8] = {&xa.x, &xa.y, &xa.z, &xa.w, &xb.x, &xb.y, &xb.z, &xb.w};
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                *xv[2 * m] += (ar * p[m].re - ai * p[m].im) + (wr * sv[m].re - wi * sv[m].im);
                *xv[2 * m + 1] += (ar * p[m].im + ai * p[m].re) + (wr * sv[m].im + wi * sv[m].re);
                const float rr = sv[m].re - (wr * t[m].re - wi * t[m].im);
                const float ri = sv[m].im - (wr * t[m].im + wi * t[m].re);
                rn[4 * c + m].re = rr; rn[4 * c + m].im = ri;
                s0 += q[m].re * rr + q[m].im * ri;
                s1 += q[m].re * ri - q[m].im * rr;
                s2 += rr * rr + ri * ri;
            }
            X[(size_t)(b * 6 + 2 * c) * G.rbn + e] = xa;
            X[(size_t)(b * 6 + 2 * c + 1) * G.rbn + e] = xb;
        }
        s[0] += (double)s0; s[1] += (double)s1; s[2] += (double)s2;
        h16_store(Rr, G.rbn, e, rn);
    }
    reduce_finalize<3, K_RHO_REL>(s, G.n, rb);
}

// r = R64_i / scale_i in H16.  INIT: also r~ = r, p = v = 0, x = 0, rho = |r|^2 (K_INIT_RHO).  Otherwise (reliable update):
// r replaces the recursive residual, <r~, r> and |r|^2 feed K_REPLACE.
template <bool INIT>
__global__ void h16_demote(Geo G, RedBuf rb, const double2* __restrict__ R64, float4* __restrict__ r16, float4* __restrict__ rt16,
                           float4* __restrict__ p16, float4* __restrict__ v16, float4* __restrict__ x32) {
    WD_H16_PROLOGUE
    const double* scal = rb.scal;
    const double sc = scal[S_SCALE * WD_MAX_RHS + r];
    const double inv = sc > 0.0 ? 1.0 / sc : 0.0;
    double s[3] = {0.0, 0.0, 0.0};
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + k * stride;
        uint32_t b, e;
        locate(G, i, &b, &e);
        cx<float> a[12];
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            const double2 d = R64[(size_t)(b * 12 + c) * G.rbn + e];
            a[c].re = (float)(d.x * inv); a[c].im = (float)(d.y * inv);
        }
        h16_store(r16 + (size_t)b * G.rowH, G.rbn, e, a);
        // what the solver will see is the ROUNDED r: read it back through the format for the inner products
        cx<float> ar[12];
        h16_load<false>(r16 + (size_t)b * G.rowH, G.rbn, e, ar);
        if (INIT) {
            h16_store(rt16 + (size_t)b * G.rowH, G.rbn, e, a);
            cx<float> z[12];
#pragma unroll
            for (int c = 0; c < 12; ++c) { z[c].re = 0.f; z[c].im = 0.f; }
            h16_store(p16 + (size_t)b * G.rowH, G.rbn, e, z);
            h16_store(v16 + (size_t)b * G.rowH, G.rbn, e, z);
            store32(x32, G, b, e, z);
            float s2 = 0.f;
#pragma unroll
            for (int c = 0; c < 12; ++c) s2 += ar[c].re * ar[c].re + ar[c].im * ar[c].im;
            s[0] += (double)s2; s[2] += (double)s2;
        } else {
            cx<float> q[12];
            h16_load<false>(rt16 + (size_t)b * G.rowH, G.rbn, e, q);
            float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
            for (int c = 0; c < 12; ++c) {
                s0 += q[c].re * ar[c].re + q[c].im * ar[c].im;
                s1 += q[c].re * ar[c].im - q[c].im * ar[c].re;
                s2 += ar[c].re * ar[c].re + ar[c].im * ar[c].im;
            }
            s[0] += (double)s0; s[1] += (double)s1; s[2] += (double)s2;
        }
    }
    if (INIT) reduce_finalize<3, K_INIT_RHO>(s, G.n, rb);
    else reduce_finalize<3, K_REPLACE>(s, G.n, rb);
}

// Y_i += scale_i x_i (fp32 -> fp64), x = 0
__global__ void h16_flush(Geo G, const double* __restrict__ scal, float4* __restrict__ x32, double2* __restrict__ Y64) {
    WD_H16_PROLOGUE
    const double sc = scal[S_SCALE * WD_MAX_RHS + r];
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + k * stride;
        uint32_t b, e;
        locate(G, i, &b, &e);
        cx<float> x[12];
        load32(x32, G, b, e, x);
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            double2 y = Y64[(size_t)(b * 12 + c) * G.rbn + e];
            y.x += sc * (double)x[c].re; y.y += sc * (double)x[c].im;
            Y64[(size_t)(b * 12 + c) * G.rbn + e] = y;
            x[c].re = 0.f; x[c].im = 0.f;
        }
        store32(x32, G, b, e, x);
    }
}

// |phi_i|^2 over a full-lattice fp64 block; R = B - W (W nullable), |R_i|^2 -> K_OUT_R2_REL
__global__ void rel_norm2_kernel(long nvec, int n, RedBuf rb, const double2* __restrict__ A) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 a = A[i];
        s[0] += a.x * a.x + a.y * a.y;
    }
    reduce_finalize<1, K_PHI2>(s, n, rb);
}
__global__ void rel_resid_kernel(long nvec, int n, RedBuf rb, const double2* __restrict__ Bv, const double2* W, double2* R) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        double2 b = Bv[i];
        if (W) { const double2 w = W[i]; b.x -= w.x; b.y -= w.y; }
        R[i] = b;
        s[0] += b.x * b.x + b.y * b.y;
    }
    reduce_finalize<1, K_OUT_R2_REL>(s, n, rb);
}

__global__ void rel_set_globals(double* scal, double tol2, double delta2) {
    scal[G_TOL2] = tol2;
    scal[G_DELTA2] = delta2;
    scal[G_DONE] = 0.0;
    scal[G_ITERS] = 0.0;
    scal[G_OUT_DONE] = 0.0;
    scal[G_UPDATES] = 0.0;
}

void shape(const wd_ctx* c, long work, int n, int* B, unsigned* G) {
    const int m = (8 + n - 1) / n;
    *B = 32 * n * m;
    long g = (work + *B - 1) / *B;
    const long cap = (long)c->n_sm * 4;
    *G = (unsigned)(g < cap ? (g < 1 ? 1 : g) : cap);
}

}  // namespace

// The 16-bit route runs only where the z-march hop kernel takes H16 operands in this link form: row-major layout,
// Lx/2 * n a multiple of 4, and a CTA shape that fits (Lx/2 * n consumer threads + the producer warps <= 512, so e.g.
// not Lx = 64 at n = 16).  Elsewhere wd_solve_impl runs the default solver, as include/wd.h promises.
bool wd_solve_h16_applies(const wd_ctx* c, int recon, int n) {
    return n >= 3 && wd_hop_zm_serves(c, recon, n, 1);
}

size_t wd_h16_half_bytes(const wd_ctx* c, int n) { return (size_t)c->Vh * n * 52; }

// delta = inner_tol (0 -> 0.1): a reliable update when |r_i| < delta * max |r_i| since the last one
int wd_solve_h16(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_updates, int max_iters,
                 double delta, int recon, wd_solve_info* info) {
    const auto t_begin = std::chrono::steady_clock::now();
    cudaStream_t st = c->stream;
    const long Vh = c->Vh;
    const size_t hb64 = wd_half_bytes(c, WD_F64, n);
    const size_t sb64 = wd_align_up(wd_half_bytes(c, WD_F64, c->max_rhs)), sb32 = wd_align_up(wd_half_bytes(c, WD_F32, c->max_rhs));
    // the same scratch map as wd_solve_impl: three fp64 blocks, then seven fp32-sized slots (an H16 block fits in one)
    char* w = c->d_solver;
    double2* phihat = (double2*)w; w += sb64;
    double2* tmp64 = (double2*)w;  w += sb64;
    double2* R64 = (double2*)w;    w += sb64;
    float4* x32 = (float4*)w;   w += sb32;
    float4* r16 = (float4*)w;   w += sb32;
    float4* p16 = (float4*)w;   w += sb32;
    float4* v16 = (float4*)w;   w += sb32;
    float4* t16 = (float4*)w;   w += sb32;
    float4* rt16 = (float4*)w;  w += sb32;
    float4* tmp16 = (float4*)w; w += sb32;

    const char* PhiE = (const char*)Phi;
    const char* PhiO = PhiE + hb64;
    char* XE = (char*)X;
    char* XO = XE + hb64;
    const double kap = c->kappa;
    RedBuf rb{c->d_scal, c->d_partials, c->d_ticket, c->d_hist, c->hist_cap};
    int rc;
    Geo G;
    G.items = Vh * n; G.RB = c->RB; G.n = (uint32_t)n; G.rbn = c->RB * (uint32_t)n; G.rowH = h16_row_vecs(G.rbn);

    { wd_prof_scope pr__(c, WD_PROF_BLAS); rel_set_globals<<<1, 1, 0, st>>>(c->d_scal, tol * tol, delta * delta); }
    WD_LAUNCH_CHECK(c);
    const long nv64 = 12 * Vh * n;
    int B64, Bi; unsigned G64, G64f, Gi;
    shape(c, nv64, n, &B64, &G64);
    shape(c, 2 * nv64, n, &B64, &G64f);
    shape(c, G.items, n, &Bi, &Gi);

    { wd_prof_scope pr__(c, WD_PROF_BLAS); rel_norm2_kernel<<<G64f, B64, 0, st>>>(2 * nv64, n, rb, (const double2*)Phi); }
    WD_LAUNCH_CHECK(c);
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, PhiO, phihat, PhiE, 1.0, kap);
    if (rc) return rc;
    WD_CUDA_CHECK(c, cudaMemsetAsync(XE, 0, hb64, st));
    { wd_prof_scope pr__(c, WD_PROF_BLAS); rel_resid_kernel<<<G64, B64, 0, st>>>(nv64, n, rb, phihat, nullptr, R64); }
    WD_LAUNCH_CHECK(c);
    double* hp = c->h_pinned;
    WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
    WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
    int converged = hp[G_OUT_DONE] != 0.0 ? 1 : 0, updates = 0;
    if (!converged) {
        { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_demote<true><<<Gi, Bi, 0, st>>>(G, rb, R64, r16, rt16, p16, v16, x32); }
        WD_LAUNCH_CHECK(c);
        const int poll_every = c->opt[WD_OPT_POLL_EVERY];
        int sweep_dir = 0;
        auto sweep = [&]() { sweep_dir ^= c->opt[WD_OPT_ALTERNATE_SWEEP] ? 1 : 0; return sweep_dir; };
        wd_hop_ops o;
        o.check_done = true;
        o.storage = 1;
        int it = 0;
        while (it < max_iters) {
            ++it;
            { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_p_update<<<Gi, Bi, 0, st>>>(G, sweep(), c->d_scal, r16, p16, v16); }
            WD_LAUNCH_CHECK(c);
            o.in = p16; o.out = tmp16; o.in2 = nullptr; o.in3 = nullptr; o.a = 0.0; o.b = 1.0; o.epi = 0; o.rev = sweep();
            rc = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 1, o);
            if (rc) return rc;
            o.in = tmp16; o.out = v16; o.in2 = p16; o.in3 = rt16; o.a = 1.0; o.b = -kap * kap; o.epi = 2; o.rev = sweep();
            rc = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 0, o);
            if (rc) return rc;
            { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_s_update<<<Gi, Bi, 0, st>>>(G, sweep(), c->d_scal, r16, v16); }
            WD_LAUNCH_CHECK(c);
            o.in = r16; o.out = tmp16; o.in2 = nullptr; o.in3 = nullptr; o.a = 0.0; o.b = 1.0; o.epi = 0; o.rev = sweep();
            rc = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 1, o);
            if (rc) return rc;
            o.in = tmp16; o.out = t16; o.in2 = r16; o.in3 = nullptr; o.a = 1.0; o.b = -kap * kap; o.epi = 3; o.rev = sweep();
            rc = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 0, o);
            if (rc) return rc;
            { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_xr_update<<<Gi, Bi, 0, st>>>(G, sweep(), rb, x32, p16, r16, t16, rt16); }
            WD_LAUNCH_CHECK(c);
            if (it % poll_every != 0 && it != max_iters) continue;
            WD_CUDA_CHECK(c, cudaMemcpyAsync(hp + G_COUNT, c->d_scal + G_DONE, sizeof(double), cudaMemcpyDeviceToHost, st));
            WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
            if (hp[G_COUNT] == 0.0 && it != max_iters) continue;
            // ---- reliable update: the iteration kernels have been no-ops since the flag was raised
            ++updates;
            { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_flush<<<Gi, Bi, 0, st>>>(G, c->d_scal, x32, (double2*)XE); }
            WD_LAUNCH_CHECK(c);
            rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, XE, tmp64, nullptr, 0.0, 1.0);
            if (rc) return rc;
            rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, tmp64, R64, XE, 1.0, -kap * kap);
            if (rc) return rc;
            { wd_prof_scope pr__(c, WD_PROF_BLAS); rel_resid_kernel<<<G64, B64, 0, st>>>(nv64, n, rb, phihat, R64, R64); }
            WD_LAUNCH_CHECK(c);
            { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_demote<false><<<Gi, Bi, 0, st>>>(G, rb, R64, r16, rt16, p16, v16, x32); }
            WD_LAUNCH_CHECK(c);
            WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
            WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
            if (hp[G_OUT_DONE] != 0.0) { converged = 1; break; }
            if (updates >= max_updates) break;
        }
        if (!converged) {   // ran out of iterations between updates: make X the best iterate
            { wd_prof_scope pr__(c, WD_PROF_BLAS); h16_flush<<<Gi, Bi, 0, st>>>(G, c->d_scal, x32, (double2*)XE); }
            WD_LAUNCH_CHECK(c);
        }
    }
    // X_o = Phi_o + kappa H_oe X_e
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, XE, XO, PhiO, 1.0, kap);
    if (rc) return rc;
    if (info) {
        info->n_rhs = n;
        info->outer_steps = updates;
        info->inner_iters_total = (int)hp[G_ITERS];
        info->converged = converged;
        for (int r = 0; r < n; ++r) {
            const double phi2 = hp[S_PHI2 * WD_MAX_RHS + r], r2 = hp[S_OUT_R2 * WD_MAX_RHS + r];
            info->bnorm[r] = sqrt(phi2);
            info->relres[r] = phi2 > 0.0 ? sqrt(r2 / phi2) : 0.0;
        }
        for (int r = n; r < WD_MAX_RHS; ++r) info->bnorm[r] = info->relres[r] = 0.0;
        info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
    }
    return converged ? WD_OK : WD_ENOCONV;
}
