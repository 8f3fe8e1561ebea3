// wd_solve.cu -- blocked mixed-precision solve (hot-path steps a1, a3-a7).
//
//   A X = Phi,  A = D or D^dag, all n_rhs columns in lock-step.
//   even/odd:  Ahat = 1 - kappa^2 H_eo H_oe on even sites,
//        Phihat_e = Phi_e + kappa H_eo Phi_o,   Ahat X_e = Phihat_e,   X_o = Phi_o + kappa H_oe X_e.
//   outer loop, fp64 (defect correction, the "mixed-precision preconditioner technique" of
//   PAPER.md:80-82 in its simplest form; reading R11):
//        R = Phihat_e - Ahat X_e;  stop when |R_i| <= tol |phi_i| for every i;
//        E = BiCGStab_fp32(R_i / |R_i|);  X_e,i += |R_i| E_i.
//   inner loop, fp32: textbook BiCGStab per column, per-column alpha, beta, omega kept
//   on the device; a converged column is frozen (alpha = omega = beta = 0).
#include <chrono>

#include "wd_blas.cuh"

using namespace wdblas;

namespace {

// 128-bit element -> its two complex numbers (re, im, re, im).  PAIRED: the element is in the P32 form of wd_f2.cuh,
// (A.re, B.re, A.im, B.im); both lanes belong to the same column, so the per-column scalars apply to both.
template <typename T, bool PAIRED>
__device__ __forceinline__ void to_arr(const typename V<T>::type& v, T (&a)[2 * V<T>::NC]);
template <> __device__ __forceinline__ void to_arr<float, false>(const float4& v, float (&a)[4]) { a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
template <> __device__ __forceinline__ void to_arr<float, true>(const float4& v, float (&a)[4]) { a[0] = v.x; a[1] = v.z; a[2] = v.y; a[3] = v.w; }
template <bool PAIRED>
__device__ __forceinline__ float4 from_arr(const float (&a)[4]) {
    return PAIRED ? make_float4(a[0], a[2], a[1], a[3]) : make_float4(a[0], a[1], a[2], a[3]);
}

#define WD_BLAS_PROLOGUE(T)                                                        \
    typedef typename V<T>::type vec;                                               \
    constexpr int NC = V<T>::NC;                                                   \
    const int r = threadIdx.x % n;                                                 \
    const long stride = (long)gridDim.x * blockDim.x;                              \
    const long i0 = (long)blockIdx.x * blockDim.x + threadIdx.x;                   \
    const long cnt = i0 < nvec ? (nvec - 1 - i0) / stride + 1 : 0;

// P = R + beta (P - omega V)
template <typename T, bool PAIRED>
__global__ void p_update_kernel(long nvec, int n, int rev, const double* __restrict__ scal, const typename V<T>::type* __restrict__ R,
                                typename V<T>::type* __restrict__ P, const typename V<T>::type* __restrict__ Vv) {
    if (scal[G_DONE] != 0.0) return;
    WD_BLAS_PROLOGUE(T)
    const T br = (T)scal[S_BETA_RE * WD_MAX_RHS + r], bi = (T)scal[S_BETA_IM * WD_MAX_RHS + r];
    const T wr = (T)scal[S_OMEGA_RE * WD_MAX_RHS + r], wi = (T)scal[S_OMEGA_IM * WD_MAX_RHS + r];
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;  // rev: sweep from the top, see wd_solve_impl
        T a[2 * NC], p[2 * NC], v[2 * NC];
        to_arr<T, PAIRED>(R[i], a); to_arr<T, PAIRED>(P[i], p); to_arr<T, PAIRED>(Vv[i], v);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const T tr = p[2 * c] - (wr * v[2 * c] - wi * v[2 * c + 1]);
            const T ti = p[2 * c + 1] - (wr * v[2 * c + 1] + wi * v[2 * c]);
            p[2 * c] = a[2 * c] + (br * tr - bi * ti);
            p[2 * c + 1] = a[2 * c + 1] + (br * ti + bi * tr);
        }
        P[i] = from_arr<PAIRED>(p);
    }
}

// S = R - alpha V   (in place on R)
template <typename T, bool PAIRED>
__global__ void s_update_kernel(long nvec, int n, int rev, const double* __restrict__ scal, typename V<T>::type* __restrict__ R,
                                const typename V<T>::type* __restrict__ Vv) {
    if (scal[G_DONE] != 0.0) return;
    WD_BLAS_PROLOGUE(T)
    const T ar = (T)scal[S_ALPHA_RE * WD_MAX_RHS + r], ai = (T)scal[S_ALPHA_IM * WD_MAX_RHS + r];
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;  // rev: sweep from the top, see wd_solve_impl
        T a[2 * NC], v[2 * NC];
        to_arr<T, PAIRED>(R[i], a); to_arr<T, PAIRED>(Vv[i], v);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            a[2 * c] -= ar * v[2 * c] - ai * v[2 * c + 1];
            a[2 * c + 1] -= ar * v[2 * c + 1] + ai * v[2 * c];
        }
        R[i] = from_arr<PAIRED>(a);
    }
}

// X += alpha P + omega S;  R = S - omega T;  <Rt, R>, |R|^2  ->  rho, beta, convergence flags
template <typename T, bool PAIRED>
__global__ void xr_update_kernel(long nvec, int n, int rev, RedBuf rb, typename V<T>::type* __restrict__ X,
                                 const typename V<T>::type* __restrict__ P, typename V<T>::type* __restrict__ R,
                                 const typename V<T>::type* __restrict__ Tt, const typename V<T>::type* __restrict__ Rt) {
    if (rb.scal[G_DONE] != 0.0) return;
    WD_BLAS_PROLOGUE(T)
    const double* scal = rb.scal;
    const T ar = (T)scal[S_ALPHA_RE * WD_MAX_RHS + r], ai = (T)scal[S_ALPHA_IM * WD_MAX_RHS + r];
    const T wr = (T)scal[S_OMEGA_RE * WD_MAX_RHS + r], wi = (T)scal[S_OMEGA_IM * WD_MAX_RHS + r];
    double s[3] = {0.0, 0.0, 0.0};
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;  // rev: sweep from the top, see wd_solve_impl
        T x[2 * NC], p[2 * NC], sv[2 * NC], t[2 * NC], q[2 * NC];
        to_arr<T, PAIRED>(X[i], x); to_arr<T, PAIRED>(P[i], p); to_arr<T, PAIRED>(R[i], sv); to_arr<T, PAIRED>(Tt[i], t); to_arr<T, PAIRED>(Rt[i], q);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            x[2 * c] += (ar * p[2 * c] - ai * p[2 * c + 1]) + (wr * sv[2 * c] - wi * sv[2 * c + 1]);
            x[2 * c + 1] += (ar * p[2 * c + 1] + ai * p[2 * c]) + (wr * sv[2 * c + 1] + wi * sv[2 * c]);
            const T rr = sv[2 * c] - (wr * t[2 * c] - wi * t[2 * c + 1]);
            const T ri = sv[2 * c + 1] - (wr * t[2 * c + 1] + wi * t[2 * c]);
            sv[2 * c] = rr; sv[2 * c + 1] = ri;
            s[0] += (double)q[2 * c] * rr + (double)q[2 * c + 1] * ri;
            s[1] += (double)q[2 * c] * ri - (double)q[2 * c + 1] * rr;
            s[2] += (double)rr * rr + (double)ri * ri;
        }
        X[i] = from_arr<PAIRED>(x);
        R[i] = from_arr<PAIRED>(sv);
    }
    reduce_finalize<3, K_RHO>(s, n, rb);
}

// The merged update (WD_OPT_MERGE): X += alpha P + omega S;  R = S - omega T;  P = R + beta (P - omega V);  |R|^2.
// beta = (rho'/rho)(alpha/omega) is already on the device: rho' = <Rt,S> - omega <Rt,T> came out of the epilogue of the
// hop that made T (K_OMEGA_RHO), so the new P can be formed in the same pass as the new R.  5 reads + 3 writes.
template <typename T, bool PAIRED>
__global__ void xrp_update_kernel(long nvec, int n, int rev, RedBuf rb, typename V<T>::type* __restrict__ X,
                                  typename V<T>::type* __restrict__ P, typename V<T>::type* __restrict__ R,
                                  const typename V<T>::type* __restrict__ Tt, const typename V<T>::type* __restrict__ Vv) {
    if (rb.scal[G_DONE] != 0.0) return;
    WD_BLAS_PROLOGUE(T)
    const double* scal = rb.scal;
    const T ar = (T)scal[S_ALPHA_RE * WD_MAX_RHS + r], ai = (T)scal[S_ALPHA_IM * WD_MAX_RHS + r];
    const T wr = (T)scal[S_OMEGA_RE * WD_MAX_RHS + r], wi = (T)scal[S_OMEGA_IM * WD_MAX_RHS + r];
    const T br = (T)scal[S_BETA_RE * WD_MAX_RHS + r], bi = (T)scal[S_BETA_IM * WD_MAX_RHS + r];
    double s[1] = {0.0};
    for (long k = 0; k < cnt; ++k) {
        const long i = i0 + (rev ? cnt - 1 - k : k) * stride;
        T x[2 * NC], p[2 * NC], sv[2 * NC], t[2 * NC], v[2 * NC];
        to_arr<T, PAIRED>(X[i], x); to_arr<T, PAIRED>(P[i], p); to_arr<T, PAIRED>(R[i], sv); to_arr<T, PAIRED>(Tt[i], t); to_arr<T, PAIRED>(Vv[i], v);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            x[2 * c] += (ar * p[2 * c] - ai * p[2 * c + 1]) + (wr * sv[2 * c] - wi * sv[2 * c + 1]);
            x[2 * c + 1] += (ar * p[2 * c + 1] + ai * p[2 * c]) + (wr * sv[2 * c + 1] + wi * sv[2 * c]);
            const T rr = sv[2 * c] - (wr * t[2 * c] - wi * t[2 * c + 1]);
            const T ri = sv[2 * c + 1] - (wr * t[2 * c + 1] + wi * t[2 * c]);
            const T tr = p[2 * c] - (wr * v[2 * c] - wi * v[2 * c + 1]);
            const T ti = p[2 * c + 1] - (wr * v[2 * c + 1] + wi * v[2 * c]);
            sv[2 * c] = rr; sv[2 * c + 1] = ri;
            p[2 * c] = rr + (br * tr - bi * ti);
            p[2 * c + 1] = ri + (br * ti + bi * tr);
            s[0] += (double)rr * rr + (double)ri * ri;
        }
        X[i] = from_arr<PAIRED>(x);
        R[i] = from_arr<PAIRED>(sv);
        P[i] = from_arr<PAIRED>(p);
    }
    reduce_finalize<1, K_RNORM>(s, n, rb);
}

// |phi_i|^2 over a full-lattice fp64 block
__global__ void norm2_kernel(long nvec, int n, RedBuf rb, const double2* __restrict__ A) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 a = A[i];
        s[0] += a.x * a.x + a.y * a.y;
    }
    reduce_finalize<1, K_PHI2>(s, n, rb);
}

// R = B - W (W may be null: R = B), |R_i|^2 -> outer convergence flags, scale, inner threshold
__global__ void outer_resid_kernel(long nvec, int n, RedBuf rb, const double2* __restrict__ Bv, const double2* W,
                                   double2* R) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        double2 b = Bv[i];
        if (W) { const double2 w = W[i]; b.x -= w.x; b.y -= w.y; }
        R[i] = b;
        s[0] += b.x * b.x + b.y * b.y;
    }
    reduce_finalize<1, K_OUT_R2>(s, n, rb);
}

// inner start: b = R_i / |R_i| in fp32 -> r, rt;  x = p = v = 0;  rho = <b, b>.
// fp64 vec index ((block*12 + k)*RB + o)*n + r, k < 12  <->  fp32 vec index ((block*6 + k/2)*RB + o)*n + r, components 2*(k%2)..
// PAIRED: the fp32 side is P32 (wd_f2.cuh): vec index ((block*12 + k)*H + p)*n + r = complex k of sites o = p and p + H, H = RB/2.
// P_IS_R (merged-update schedule): p starts as r, because no p-update precedes the first hop there.
template <bool PAIRED, bool P_IS_R = false>
__global__ void demote_kernel(long Vh, long RB, int n, RedBuf rb, const double2* __restrict__ R64, float4* __restrict__ r32,
                              float4* __restrict__ rt32, float4* __restrict__ x32, float4* __restrict__ p32,
                              float4* __restrict__ v32) {
    const int r = threadIdx.x % n;
    const long stride = (long)gridDim.x * blockDim.x;
    const long nvec = 6 * Vh * n, half = RB * n;  // i / half = block * 6 + c  <->  fp64 chunks 2 (block * 6 + c), + 1
    const double* scal = rb.scal;
    const bool frozen = scal[S_FLAG * WD_MAX_RHS + r] != 0.0;
    const double sc = scal[S_SCALE * WD_MAX_RHS + r];
    const double inv = (frozen || !(sc > 0.0)) ? 0.0 : 1.0 / sc;
    double s[3] = {0.0, 0.0, 0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        double2 a, b;
        if (PAIRED) {   // i = bk * (half/2) + rem, bk = block*12 + k:  lane A at fp64 index bk*half + rem, lane B half/2 further
            const long bk = i / (half / 2), rem = i - bk * (half / 2);
            const double2 sa = R64[bk * half + rem], sb = R64[bk * half + half / 2 + rem];
            a = make_double2(sa.x, sb.x); b = make_double2(sa.y, sb.y);
        } else {
            const long c = i / half, rem = i - c * half;
            a = R64[(2 * c) * half + rem]; b = R64[(2 * c + 1) * half + rem];
        }
        const float4 f = make_float4((float)(a.x * inv), (float)(a.y * inv), (float)(b.x * inv), (float)(b.y * inv));
        r32[i] = f;
        rt32[i] = f;
        const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
        x32[i] = z; p32[i] = P_IS_R ? f : z; v32[i] = z;
        s[0] += (double)f.x * f.x + (double)f.y * f.y + (double)f.z * f.z + (double)f.w * f.w;
    }
    s[2] = s[0];
    reduce_finalize<3, K_INIT_RHO>(s, n, rb);
}

// X_i += |R_i| E_i  (fp32 -> fp64)
template <bool PAIRED>
__global__ void promote_kernel(long Vh, long RB, int n, const double* __restrict__ scal, const float4* __restrict__ e32,
                               double2* __restrict__ X64) {
    const int r = threadIdx.x % n;
    const long stride = (long)gridDim.x * blockDim.x;
    const long nvec = 6 * Vh * n, half = RB * n;  // i / half = block * 6 + c  <->  fp64 chunks 2 (block * 6 + c), + 1
    const double sc = scal[S_OUT_CONV * WD_MAX_RHS + r] != 0.0 ? 0.0 : scal[S_SCALE * WD_MAX_RHS + r];
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const float4 f = e32[i];
        if (PAIRED) {
            const long bk = i / (half / 2), rem = i - bk * (half / 2);
            double2 a = X64[bk * half + rem], b = X64[bk * half + half / 2 + rem];
            a.x += sc * f.x; b.x += sc * f.y; a.y += sc * f.z; b.y += sc * f.w;
            X64[bk * half + rem] = a;
            X64[bk * half + half / 2 + rem] = b;
        } else {
            const long c = i / half, rem = i - c * half;
            double2 a = X64[(2 * c) * half + rem], b = X64[(2 * c + 1) * half + rem];
            a.x += sc * f.x; a.y += sc * f.y; b.x += sc * f.z; b.y += sc * f.w;
            X64[(2 * c) * half + rem] = a;
            X64[(2 * c + 1) * half + rem] = b;
        }
    }
}

__global__ void set_globals_kernel(double* scal, double tol2, double intol2) {
    scal[G_TOL2] = tol2;
    scal[G_INTOL2] = intol2;
    scal[G_DONE] = 0.0;
    scal[G_ITERS] = 0.0;
    scal[G_OUT_DONE] = 0.0;
}

struct Launch {
    int B;
    unsigned G;
};
Launch blas_cfg(const wd_ctx* c, long nvec, int n) {
    Launch l;
    const int m = (8 + n - 1) / n;
    l.B = 32 * n * m;
    long g = (nvec + l.B - 1) / l.B;
    const long cap = (long)c->n_sm * 4;
    l.G = (unsigned)(g < cap ? (g < 1 ? 1 : g) : cap);
    return l;
}

}  // namespace

size_t wd_solver_scratch_bytes(const wd_ctx* c) {
    const int n = c->max_rhs;
    size_t b = 0;
    b += 3 * wd_align_up(wd_half_bytes(c, WD_F64, n));      // phihat, tmp_o, R/W
    b += 7 * wd_align_up(wd_half_bytes(c, WD_F32, n));      // x, r, p, v, t, rt, tmp_o
    b += 8 * wd_align_up(wd_half_bytes(c, WD_F64, n));      // blocked outer solvers (wd_solve_gl.cu): Rt, P, V, S, T, Ph, Sh, Pnew
    b += 4 * wd_align_up(2 * wd_half_bytes(c, WD_F64, n));  // host path: canonical Phi, native Phi, X, Y
    b += wd_align_up(sizeof(double) * 4 * c->V * 18);       // host path: F
    return b;
}

// The fp32 inner solver on its own: E_i = BiCGStab_fp32(R_i / scale_i) for the columns whose S_FLAG is 0, to a recursive
// residual of S_THR2 (relative to the unit-norm right-hand side), then Xacc_i += scale_i E_i.  S_SCALE, S_FLAG, S_THR2 and
// S_OUT_CONV are set on the device by the caller's preceding reduction.  Uses the seven fp32 slots of the solver scratch.
void wd_inner_forms(const wd_ctx* c, int recon, int n, bool* paired, bool* merged) {
    const int impl = c->opt[WD_OPT_HOP_IMPL];
    // P32 (two sites per thread, packed fp32 instructions: wd_f2.cuh) wherever the z-march kernel serves it
    *paired = c->opt[WD_OPT_PAIRED] != 0 && impl >= 2 && n >= 3 && wd_hop_zm_serves(c, recon, n, 2);
    // merged x,r,p update (WD_OPT_MERGE) wherever the z-march kernel, which has the seven-sum epilogue, serves the hop
    *merged = c->opt[WD_OPT_MERGE] != 0 && !*paired && n >= 3 &&
              ((impl == 2 && wd_hop_zm_preferred(c, recon, n)) || (impl == 3 && wd_hop_zm_serves(c, recon, n, 0)));
}

int wd_inner_solve_f32(wd_ctx* c, int dag, int n, int recon, int max_inner, const double2* R64, double2* Xacc) {
    cudaStream_t st = c->stream;
    const long Vh = c->Vh;
    const size_t sb64 = wd_align_up(wd_half_bytes(c, WD_F64, c->max_rhs)), sb32 = wd_align_up(wd_half_bytes(c, WD_F32, c->max_rhs));
    char* w = c->d_solver + 3 * sb64;
    float4* x32 = (float4*)w;   w += sb32;
    float4* r32 = (float4*)w;   w += sb32;
    float4* p32 = (float4*)w;   w += sb32;
    float4* v32 = (float4*)w;   w += sb32;
    float4* t32 = (float4*)w;   w += sb32;
    float4* rt32 = (float4*)w;  w += sb32;
    float4* tmp32 = (float4*)w; w += sb32;
    const double kap = c->kappa;
    RedBuf rb{c->d_scal, c->d_partials, c->d_ticket, c->d_hist, c->hist_cap};
    const long nv32 = 6 * Vh * n;
    const Launch L32 = blas_cfg(c, nv32, n);
    // Schroedinger functional, row-major layout: the rows of the frozen t = 0 slice open every half-lattice block and hold
    // zeros in every vector of the solver (the demotion writes them, the hops keep them); the update kernels of the
    // iteration skip them: 1/T of their bytes
    const long skip = (c->bc == WD_BC_SF && c->order == WD_ORDER_LINEAR && c->RB == (uint32_t)(c->L[0] / 2))
                          ? (long)c->L[1] * c->L[2] * 6 * (c->L[0] / 2) * n : 0;
    const long nvu = nv32 - skip;
    const Launch LU = blas_cfg(c, nvu, n);
    float4 *xu = x32 + skip, *ru = r32 + skip, *pu = p32 + skip, *vu = v32 + skip, *tu = t32 + skip, *rtu = rt32 + skip;
    double* hp = c->h_pinned;
    int rc;
    {
        // P32 (two sites per thread, packed fp32 instructions: wd_f2.cuh) wherever the z-march kernel serves it
        bool paired, merged;
        wd_inner_forms(c, recon, n, &paired, &merged);
        {
            wd_prof_scope pr__(c, WD_PROF_BLAS);
            if (paired) demote_kernel<true><<<L32.G, L32.B, 0, st>>>(Vh, (long)c->RB, n, rb, R64, r32, rt32, x32, p32, v32);
            else if (merged) demote_kernel<false, true><<<L32.G, L32.B, 0, st>>>(Vh, (long)c->RB, n, rb, R64, r32, rt32, x32, p32, v32);
            else demote_kernel<false><<<L32.G, L32.B, 0, st>>>(Vh, (long)c->RB, n, rb, R64, r32, rt32, x32, p32, v32);
        }
        WD_LAUNCH_CHECK(c);
        // One iteration = 3 BLAS1 kernels + 4 hops; sigma and omega are reduced inside the even-parity hops.
        // Kernels turn into no-ops once the device-side done flag is set, so iterations are enqueued
        // poll_every at a time and the host only looks at the flag in between.
        const int poll_every = c->opt[WD_OPT_POLL_EVERY];
        // Consecutive kernels sweep the vectors in opposite directions: what one kernel wrote last (and the
        // 126 MB L2 still holds) is what the next one reads first.
        int sweep_dir = 0;
        auto sweep = [&]() { sweep_dir ^= c->opt[WD_OPT_ALTERNATE_SWEEP] ? 1 : 0; return sweep_dir; };
        wd_hop_ops o;
        o.check_done = true;
        o.storage = paired ? 2 : 0;
        // one BiCGStab iteration on c->stream (which is the capture stream while a graph is being recorded)
        auto enqueue_iteration = [&]() -> int {
            if (!merged) {
                wd_prof_scope pr__(c, WD_PROF_BLAS);
                if (paired) p_update_kernel<float, true><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), c->d_scal, ru, pu, vu);
                else p_update_kernel<float, false><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), c->d_scal, ru, pu, vu);
                WD_LAUNCH_CHECK(c);
            }
            // v = Ahat p, sigma = <rt, v> -> alpha.  (wd_profile: one event pair brackets the two hop launches of an
            // application of Ahat, so that the per-launch average carries one kernel-to-kernel gap, not two.)
            int rc2;
            {
                wd_prof_scope pr__(c, WD_PROF_HOP32);
                o.in = p32; o.out = tmp32; o.in2 = nullptr; o.in3 = nullptr; o.a = 0.0; o.b = 1.0; o.epi = 0;
                o.rev = sweep();
                rc2 = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 1, o);
                if (rc2) return rc2;
                o.in = tmp32; o.out = v32; o.in2 = p32; o.in3 = rt32; o.a = 1.0; o.b = -kap * kap; o.epi = 2;
                o.rev = sweep();
                rc2 = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 0, o);
                if (rc2) return rc2;
            }
            {
                wd_prof_scope pr__(c, WD_PROF_BLAS);
                if (paired) s_update_kernel<float, true><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), c->d_scal, ru, vu);
                else s_update_kernel<float, false><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), c->d_scal, ru, vu);
            }
            WD_LAUNCH_CHECK(c);
            // t = Ahat s, <t, s>, <t, t> -> omega
            {
                wd_prof_scope pr__(c, WD_PROF_HOP32);
                o.in = r32; o.out = tmp32; o.in2 = nullptr; o.in3 = nullptr; o.a = 0.0; o.b = 1.0; o.epi = 0;
                o.rev = sweep();
                rc2 = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 1, o);
                if (rc2) return rc2;
                o.in = tmp32; o.out = t32; o.in2 = r32; o.in3 = merged ? rt32 : nullptr; o.a = 1.0; o.b = -kap * kap; o.epi = merged ? 4 : 3;
                o.rev = sweep();
                rc2 = wd_hop_launch_ex(c, WD_F32, recon, dag, n, 0, o);
                if (rc2) return rc2;
            }
            {
                wd_prof_scope pr__(c, WD_PROF_BLAS);
                if (merged) xrp_update_kernel<float, false><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), rb, xu, pu, ru, tu, vu);
                else if (paired) xr_update_kernel<float, true><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), rb, xu, pu, ru, tu, rtu);
                else xr_update_kernel<float, false><<<LU.G, LU.B, 0, c->stream>>>(nvu, n, sweep(), rb, xu, pu, ru, tu, rtu);
            }
            WD_LAUNCH_CHECK(c);
            return WD_OK;
        };
        // `iters` iterations and the read-back of the done flag
        auto enqueue_block = [&](int iters) -> int {
            for (int k = 0; k < iters; ++k) {
                const int rc2 = enqueue_iteration();
                if (rc2) return rc2;
            }
            WD_CUDA_CHECK(c, cudaMemcpyAsync(hp + G_COUNT, c->d_scal + G_DONE, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            return WD_OK;
        };
        // Full blocks are replayed as a CUDA graph (less idle time between the ~30 short dependent kernels of a block:
        // 56.2 us against 58.7 us per back-to-back hop launch at 24^4; several times that on the launch-bound small
        // lattices).  A block is a function of (operator, n_rhs, link form, the sweep direction it starts with) and of
        // the options, which clear the cache when they change.  First sight of a key: stream order (this also sets the
        // kernels' function attributes outside any capture); second: capture on the library's own stream, then replay.
        const bool use_graph = c->opt[WD_OPT_GRAPH] != 0;
        for (int it = 0; it < max_inner;) {
            const int blk = poll_every < max_inner - it ? poll_every : max_inner - it;
            const int start_dir = sweep_dir;
            bool launched = false;
            unsigned long long graph_key = 0;
            if (use_graph && blk == poll_every) {
                const unsigned long long key = graph_key = (unsigned long long)dag | ((unsigned long long)n << 1) | ((unsigned long long)recon << 8) |
                                               ((unsigned long long)start_dir << 9) | ((unsigned long long)(paired ? 1 : 0) << 10) |
                                               ((unsigned long long)(c->prof_on ? 1 : 0) << 11) | ((unsigned long long)(merged ? 1 : 0) << 12);
                wd_graph_entry* ge = nullptr;
                for (wd_graph_entry& g : c->graphs)
                    if (g.key == key) ge = &g;
                if (ge == nullptr) {
                    c->graphs.push_back(wd_graph_entry{key, nullptr, 0, {}, {}});
                } else {
                    if (ge->exec == nullptr) {
                        if (!c->cap_stream) WD_CUDA_CHECK(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
                        cudaStream_t user = c->stream;
                        const long long l0 = c->launches;
                        WD_CUDA_CHECK(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed));
                        c->stream = c->cap_stream;
                        c->prof_graph = ge;
                        rc = enqueue_block(blk);
                        c->prof_graph = nullptr;
                        c->stream = user;
                        cudaGraph_t graph = nullptr;
                        const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
                        ge->launches = c->launches - l0;
                        c->launches = l0;
                        sweep_dir = start_dir;
                        if (rc != WD_OK || e != cudaSuccess) {
                            if (graph) cudaGraphDestroy(graph);
                            if (rc != WD_OK) return rc;
                            c->err = std::string("graph capture: ") + cudaGetErrorString(e);
                            return WD_ECUDA;
                        }
                        const cudaError_t e2 = cudaGraphInstantiate(&ge->exec, graph, 0);
                        cudaGraphDestroy(graph);
                        if (e2 != cudaSuccess) {
                            ge->exec = nullptr;
                            c->err = std::string("graph instantiate: ") + cudaGetErrorString(e2);
                            return WD_ECUDA;
                        }
                    }
                    WD_CUDA_CHECK(c, cudaGraphLaunch(ge->exec, c->stream));
                    c->launches += ge->launches;
                    if (c->opt[WD_OPT_ALTERNATE_SWEEP] && (((merged ? 6 : 7) * blk) & 1)) sweep_dir ^= 1;   // launches per iteration
                    launched = true;
                }
            }
            if (!launched) {
                rc = enqueue_block(blk);
                if (rc) return rc;
            }
            it += blk;
            WD_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
            if (launched && c->prof_on) {   // the replay's event pairs: add them up before the next replay re-records them
                for (wd_graph_entry& g : c->graphs) {
                    if (g.key != graph_key) continue;
                    for (size_t e = 0; e < g.cls.size(); ++e) {
                        float t = 0.f;
                        if (cudaEventElapsedTime(&t, g.ev[2 * e], g.ev[2 * e + 1]) == cudaSuccess) {
                            c->prof_acc_ms[g.cls[e]] += t;
                            c->prof_acc_cnt[g.cls[e]] += 1;
                        }
                    }
                }
            }
            if (hp[G_COUNT] != 0.0) break;
        }
        {
            wd_prof_scope pr__(c, WD_PROF_BLAS);
            if (paired) promote_kernel<true><<<L32.G, L32.B, 0, st>>>(Vh, (long)c->RB, n, c->d_scal, x32, Xacc);
            else promote_kernel<false><<<L32.G, L32.B, 0, st>>>(Vh, (long)c->RB, n, c->d_scal, x32, Xacc);
        }
        WD_LAUNCH_CHECK(c);
    }
    return WD_OK;
}

// Solver dispatch (WD_OPT_SOLVER).  inner_tol = 0 picks each solver's default.
int wd_solve_impl(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_outer,
                  int max_inner, double inner_tol, int recon, wd_solve_info* info) {
    const int solver = c->opt[WD_OPT_SOLVER];
    if (solver == WD_SOLVER_GL_FLEX || solver == WD_SOLVER_GL_F64)
        return wd_solve_gl(c, solver == WD_SOLVER_GL_FLEX, dag, n, Phi, X, tol, max_outer, max_inner, inner_tol > 0.0 ? inner_tol : 1e-5,
                           recon, info);
    if (solver == WD_SOLVER_BL_F64) {
        const int rc = wd_solve_bl(c, dag, n, Phi, X, tol, max_inner, info);
        if (rc != WD_BL_BREAKDOWN) return rc;
        // rank-deficient block (zero or equal columns) or breakdown: the per-column default route solves it
    }
    if (solver == WD_SOLVER_RELIABLE_H16 && wd_solve_h16_applies(c, recon, n))
        return wd_solve_h16(c, dag, n, Phi, X, tol, max_outer, max_inner, inner_tol > 0.0 ? inner_tol : 0.01, recon, info);
    // default: the fp32 recurrence is run down to 3e-7, about what fp32 can deliver, so that TWO inner solves reach
    // 1e-12 (at 1e-5 it takes three: an fp64 residual, a demotion and a promotion more per solve; reading R12)
    return wd_solve_dc(c, dag, n, Phi, X, tol, max_outer, max_inner, inner_tol > 0.0 ? inner_tol : 3e-7, recon, info);
}

int wd_solve_dc(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_outer,
                int max_inner, double inner_tol, int recon, wd_solve_info* info) {
    const auto t_begin = std::chrono::steady_clock::now();
    cudaStream_t st = c->stream;
    const long Vh = c->Vh;
    const size_t hb64 = wd_half_bytes(c, WD_F64, n), hb32 = wd_half_bytes(c, WD_F32, n);
    const size_t sb64 = wd_align_up(wd_half_bytes(c, WD_F64, c->max_rhs)), sb32 = wd_align_up(wd_half_bytes(c, WD_F32, c->max_rhs));
    char* w = c->d_solver;
    double2* phihat = (double2*)w; w += sb64;
    double2* tmp64 = (double2*)w;  w += sb64;
    double2* R64 = (double2*)w;    w += sb64;
    float4* x32 = (float4*)w;   w += sb32;
    float4* r32 = (float4*)w;   w += sb32;
    float4* p32 = (float4*)w;   w += sb32;
    float4* v32 = (float4*)w;   w += sb32;
    float4* t32 = (float4*)w;   w += sb32;
    float4* rt32 = (float4*)w;  w += sb32;
    float4* tmp32 = (float4*)w; w += sb32;

    const char* PhiE = (const char*)Phi;
    const char* PhiO = PhiE + hb64;
    char* XE = (char*)X;
    char* XO = XE + hb64;
    const double kap = c->kappa;
    RedBuf rb{c->d_scal, c->d_partials, c->d_ticket};
    int rc;

    { wd_prof_scope pr__(c, WD_PROF_BLAS); set_globals_kernel<<<1, 1, 0, st>>>(c->d_scal, tol * tol, inner_tol * inner_tol); }
    WD_LAUNCH_CHECK(c);

    const long nv64 = 12 * Vh * n, nv32 = 6 * Vh * n;
    const Launch L64 = blas_cfg(c, nv64, n), L64f = blas_cfg(c, 2 * nv64, n), L32 = blas_cfg(c, nv32, n);

    // |phi_i|^2 (full lattice) and the even/odd right-hand side
    { wd_prof_scope pr__(c, WD_PROF_BLAS); norm2_kernel<<<L64f.G, L64f.B, 0, st>>>(2 * nv64, n, rb, (const double2*)Phi); }
    WD_LAUNCH_CHECK(c);
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, PhiO, phihat, PhiE, 1.0, kap);
    if (rc) return rc;
    WD_CUDA_CHECK(c, cudaMemsetAsync(XE, 0, hb64, st));

    int outer = 0, converged = 0;
    double* hp = c->h_pinned;
    for (;;) {
        // true residual of the even/odd system in fp64
        if (outer == 0) {
            { wd_prof_scope pr__(c, WD_PROF_BLAS); outer_resid_kernel<<<L64.G, L64.B, 0, st>>>(nv64, n, rb, phihat, nullptr, R64); }
        } else {
            rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, XE, tmp64, nullptr, 0.0, 1.0);
            if (rc) return rc;
            rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, tmp64, R64, XE, 1.0, -kap * kap);
            if (rc) return rc;
            { wd_prof_scope pr__(c, WD_PROF_BLAS); outer_resid_kernel<<<L64.G, L64.B, 0, st>>>(nv64, n, rb, phihat, R64, R64); }
        }
        WD_LAUNCH_CHECK(c);
        WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
        WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
        if (hp[G_OUT_DONE] != 0.0) { converged = 1; break; }
        if (outer >= max_outer) break;
        ++outer;

        // inner fp32 BiCGStab on the normalised residual, X_e,i += |R_i| E_i
        rc = wd_inner_solve_f32(c, dag, n, recon, max_inner, R64, (double2*)XE);
        if (rc) return rc;
    }

    // X_o = Phi_o + kappa H_oe X_e
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, XE, XO, PhiO, 1.0, kap);
    if (rc) return rc;

    if (info) {
        info->n_rhs = n;
        info->outer_steps = outer;
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
