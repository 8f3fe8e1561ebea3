// wd_solve_gl.cu -- the paper's blocked Krylov solvers as outer solvers (Table 1
// PAPER.md:110-119), alternatives to the defect-correction route of wd_solve.cu with the SAME result X = A^-1 Phi:
//
//   WD_SOLVER_GL_FLEX  (case D1)  fp64 Global BiCGStab (ref. [6]: BiCGStab on the block with Frobenius inner products, one
//       alpha, beta, omega for all columns) in its flexible form, preconditioned by the fp32 BiCGStab of wd_solve.cu run
//       per column in lock-step ("mixed-precision preconditioner"):
//           P = R + beta (P - omega V);  Ph = M(P);  V = Ahat Ph;  alpha = rho / <R~, V>_F;  S = R - alpha V;  X += alpha Ph;
//           Sh = M(S);  T = Ahat Sh;  omega = <T, S>_F / <T, T>_F;  X += omega Sh;  R = S - omega T;
//           rho' = <R~, R>_F;  beta = (rho'/rho)(alpha/omega).          M(.) ~ Ahat^-1 to inner_tol, fp32.
//       The paper reports three preconditioner calls per solve = one and a half of these iterations.
//   WD_SOLVER_GL_F64   (case B)   the same with M = identity: plain fp64 Gl-BiCGStab on the even/odd system.
//   WD_SOLVER_BL_F64   (case C)   fp64 Block BiCGStab (ref. [7]): n x n coefficient matrices from the Gram matrices
//       R~^dag V, R~^dag R, R~^dag T, second half of this file.
// The iteration stops per column on the recursive fp64 residual |r_i| <= tol |phi_i| (reading R10; reading 5 of
// "per column"); the TRUE residual phihat - Ahat X is then computed once, reported in info, and a column
// that misses tol on it restarts the recurrence from it, so "converged" means what wd_solve_block's documentation says.
#include <chrono>

#include "wd_blas.cuh"

using namespace wdblas;

namespace {

struct GlLaunch { int B; unsigned G; };
GlLaunch gl_cfg(const wd_ctx* c, long nvec, int n) {
    GlLaunch l;
    const int m = (8 + n - 1) / n;
    l.B = 32 * n * m;
    long g = (nvec + l.B - 1) / l.B;
    const long cap = (long)c->n_sm * 4;
    l.G = (unsigned)(g < cap ? (g < 1 ? 1 : g) : cap);
    return l;
}

__device__ __forceinline__ double2 cmul2(double ar, double ai, double2 b) { return make_double2(ar * b.x - ai * b.y, ar * b.y + ai * b.x); }

// |phi_i|^2 over the full lattice
__global__ void gl_norm2(long nvec, int n, RedBuf rb, const double2* __restrict__ A) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) { const double2 a = A[i]; s[0] += a.x * a.x + a.y * a.y; }
    reduce_finalize<1, K_PHI2>(s, n, rb);
}
// R = R~ = B, P = V = 0, rho = <R~, R>_F
__global__ void gl_init(long nvec, int n, RedBuf rb, const double2* __restrict__ Bv, double2* R, double2* Rt, double2* P, double2* V) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 b = Bv[i];
        R[i] = b; Rt[i] = b; P[i] = make_double2(0.0, 0.0); V[i] = make_double2(0.0, 0.0);
        s[0] += b.x * b.x + b.y * b.y;
    }
    reduce_finalize<1, K_GL_INIT>(s, n, rb);
}
// P = R + beta (P - omega V)
__global__ void gl_p_update(long nvec, const double* __restrict__ scal, const double2* __restrict__ R, double2* P, const double2* __restrict__ V) {
    const double br = scal[G_GL_BETA_RE], bi = scal[G_GL_BETA_IM], wr = scal[G_GL_OMEGA_RE], wi = scal[G_GL_OMEGA_IM];
    const long stride = (long)gridDim.x * blockDim.x;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 r = R[i], p = P[i], wv = cmul2(wr, wi, V[i]);
        const double2 t = cmul2(br, bi, make_double2(p.x - wv.x, p.y - wv.y));
        P[i] = make_double2(r.x + t.x, r.y + t.y);
    }
}
// per-column |in_i|^2 -> the inner solver's normalisation (K_PREC_PREP); out = 0
__global__ void gl_prec_prep(long nvec, int n, RedBuf rb, const double2* __restrict__ In, double2* Out) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 a = In[i];
        s[0] += a.x * a.x + a.y * a.y;
        Out[i] = make_double2(0.0, 0.0);
    }
    reduce_finalize<1, K_PREC_PREP>(s, n, rb);
}
// sigma = <R~, V>_F -> alpha
__global__ void gl_sigma(long nvec, int n, RedBuf rb, const double2* __restrict__ Rt, const double2* __restrict__ V) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[2] = {0.0, 0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 a = Rt[i], b = V[i];
        s[0] += a.x * b.x + a.y * b.y;
        s[1] += a.x * b.y - a.y * b.x;
    }
    reduce_finalize<2, K_GL_SIGMA>(s, n, rb);
}
// S = R - alpha V;  X += alpha Ph;  |S_i|^2 -> per-column convergence
__global__ void gl_s_update(long nvec, int n, RedBuf rb, const double2* __restrict__ R, const double2* __restrict__ V, double2* S,
                            double2* X, const double2* __restrict__ Ph) {
    const double ar = rb.scal[G_GL_ALPHA_RE], ai = rb.scal[G_GL_ALPHA_IM];
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 av = cmul2(ar, ai, V[i]), r = R[i], ap = cmul2(ar, ai, Ph[i]);
        const double2 sv = make_double2(r.x - av.x, r.y - av.y);
        S[i] = sv;
        double2 x = X[i];
        x.x += ap.x; x.y += ap.y;
        X[i] = x;
        s[0] += sv.x * sv.x + sv.y * sv.y;
    }
    reduce_finalize<1, K_GL_S>(s, n, rb);
}
// <T, S>_F, <T, T>_F -> omega
__global__ void gl_omega(long nvec, int n, RedBuf rb, const double2* __restrict__ T, const double2* __restrict__ S) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[3] = {0.0, 0.0, 0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 t = T[i], b = S[i];
        s[0] += t.x * b.x + t.y * b.y;
        s[1] += t.x * b.y - t.y * b.x;
        s[2] += t.x * t.x + t.y * t.y;
    }
    reduce_finalize<3, K_GL_OMEGA>(s, n, rb);
}
// X += omega Sh;  R = S - omega T;  rho' = <R~, R>_F, |R_i|^2 -> beta, convergence
__global__ void gl_xr_update(long nvec, int n, RedBuf rb, double2* X, const double2* __restrict__ Sh, double2* R, const double2* __restrict__ S,
                             const double2* __restrict__ T, const double2* __restrict__ Rt) {
    const double wr = rb.scal[G_GL_OMEGA_RE], wi = rb.scal[G_GL_OMEGA_IM];
    const long stride = (long)gridDim.x * blockDim.x;
    double s[3] = {0.0, 0.0, 0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 ws = cmul2(wr, wi, Sh[i]), wt = cmul2(wr, wi, T[i]), sv = S[i], q = Rt[i];
        double2 x = X[i];
        x.x += ws.x; x.y += ws.y;
        X[i] = x;
        const double2 r = make_double2(sv.x - wt.x, sv.y - wt.y);
        R[i] = r;
        s[0] += q.x * r.x + q.y * r.y;
        s[1] += q.x * r.y - q.y * r.x;
        s[2] += r.x * r.x + r.y * r.y;
    }
    reduce_finalize<3, K_GL_RHO>(s, n, rb);
}
// Out = Bh - AX: the true residual of the even/odd system, from which a recurrence that claims convergence is checked
// (gl_init / bl_init on it set the per-column flags) and, for the columns that miss the tolerance, restarted
__global__ void gl_true_resid(long nvec, const double2* __restrict__ Bh, const double2* __restrict__ AX, double2* __restrict__ Out) {
    const long stride = (long)gridDim.x * blockDim.x;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 b = Bh[i], a = AX[i];
        Out[i] = make_double2(b.x - a.x, b.y - a.y);
    }
}
__global__ void gl_set_globals(double* scal, double tol2, double intol2) {
    scal[G_TOL2] = tol2;
    scal[G_INTOL2] = intol2;
    scal[G_DONE] = 0.0;
    scal[G_ITERS] = 0.0;
    scal[G_OUT_DONE] = 0.0;
    scal[G_GL_BREAK] = 0.0;
}

}  // namespace

// fp64 blocks of the blocked outer solvers, behind the three fp64 and seven fp32 slots of wd_solve.cu's scratch map
static double2* gl_block(const wd_ctx* c, int k) {
    const size_t sb64 = wd_align_up(wd_half_bytes(c, WD_F64, c->max_rhs)), sb32 = wd_align_up(wd_half_bytes(c, WD_F32, c->max_rhs));
    return (double2*)(c->d_solver + 3 * sb64 + 7 * sb32 + (size_t)k * sb64);
}

// out = Ahat in = in - kappa^2 H_eo H_oe in  (fp64, two hop launches)
static int gl_apply(wd_ctx* c, int dag, int n, const double2* in, double2* tmp, double2* out) {
    int rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, in, tmp, nullptr, 0.0, 1.0);
    if (rc) return rc;
    return wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, tmp, out, in, 1.0, -c->kappa * c->kappa);
}

int wd_solve_gl(wd_ctx* c, int flex, int dag, int n, const double* Phi, double* X, double tol, int max_outer, int max_inner,
                double inner_tol, int recon, wd_solve_info* info) {
    const auto t_begin = std::chrono::steady_clock::now();
    cudaStream_t st = c->stream;
    const long Vh = c->Vh;
    const size_t hb64 = wd_half_bytes(c, WD_F64, n);
    const size_t sb64 = wd_align_up(wd_half_bytes(c, WD_F64, c->max_rhs));
    double2* phihat = (double2*)c->d_solver;
    double2* tmp64 = (double2*)(c->d_solver + sb64);
    double2* R = (double2*)(c->d_solver + 2 * sb64);
    double2 *Rt = gl_block(c, 0), *P = gl_block(c, 1), *V = gl_block(c, 2), *S = gl_block(c, 3), *T = gl_block(c, 4);
    double2 *Ph = flex ? gl_block(c, 5) : P, *Sh = flex ? gl_block(c, 6) : S;
    const char* PhiE = (const char*)Phi;
    const char* PhiO = PhiE + hb64;
    double2* XE = (double2*)X;
    char* XO = (char*)X + hb64;
    RedBuf rb{c->d_scal, c->d_partials, c->d_ticket};
    const long nv = 12 * Vh * n;
    const GlLaunch L = gl_cfg(c, nv, n), Lf = gl_cfg(c, 2 * nv, n);
    double* hp = c->h_pinned;
    int rc;
#define GL_K(call) { wd_prof_scope pr__(c, WD_PROF_BLAS); call; } WD_LAUNCH_CHECK(c)
    GL_K((gl_set_globals<<<1, 1, 0, st>>>(c->d_scal, tol * tol, inner_tol * inner_tol)));
    GL_K((gl_norm2<<<Lf.G, Lf.B, 0, st>>>(2 * nv, n, rb, (const double2*)Phi)));
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, PhiO, phihat, PhiE, 1.0, c->kappa);
    if (rc) return rc;
    WD_CUDA_CHECK(c, cudaMemsetAsync(XE, 0, hb64, st));
    GL_K((gl_init<<<L.G, L.B, 0, st>>>(nv, n, rb, phihat, R, Rt, P, V)));
    auto poll = [&]() -> int {
        WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
        WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
        return WD_OK;
    };
    // M(in) -> out: the fp32 inner solver per column (flexible form) or the identity (out aliases in)
    auto precond = [&](const double2* in, double2* out) -> int {
        if (!flex) return WD_OK;
        GL_K((gl_prec_prep<<<L.G, L.B, 0, st>>>(nv, n, rb, in, out)));
        return wd_inner_solve_f32(c, dag, n, recon, max_inner, in, out);
    };
    rc = poll();
    if (rc) return rc;
    // iteration budget: preconditioned, max_outer iterations of two preconditioner calls each (max_inner bounds every
    // inner solve); unpreconditioned there is no inner solver and max_inner bounds the iterations, as for Block BiCGStab
    const int cap = flex ? max_outer : max_inner;
    int converged = hp[G_OUT_DONE] != 0.0 ? 1 : 0, outer = 0, calls = 0;
    for (;;) {
    while (!converged && outer < cap && hp[G_GL_BREAK] == 0.0) {
        ++outer;
        GL_K((gl_p_update<<<L.G, L.B, 0, st>>>(nv, c->d_scal, R, P, V)));
        rc = precond(P, Ph);
        if (rc) return rc;
        ++calls;
        rc = gl_apply(c, dag, n, Ph, tmp64, V);
        if (rc) return rc;
        GL_K((gl_sigma<<<L.G, L.B, 0, st>>>(nv, n, rb, Rt, V)));
        GL_K((gl_s_update<<<L.G, L.B, 0, st>>>(nv, n, rb, R, V, S, XE, Ph)));
        rc = poll();
        if (rc) return rc;
        if (hp[G_OUT_DONE] != 0.0) { converged = 1; break; }   // |s_i| <= tol |phi_i| for every column: X = X + alpha Ph is the answer
        if (hp[G_GL_BREAK] != 0.0) break;
        rc = precond(S, Sh);
        if (rc) return rc;
        ++calls;
        rc = gl_apply(c, dag, n, Sh, tmp64, T);
        if (rc) return rc;
        GL_K((gl_omega<<<L.G, L.B, 0, st>>>(nv, n, rb, T, S)));
        GL_K((gl_xr_update<<<L.G, L.B, 0, st>>>(nv, n, rb, XE, Sh, R, S, T, Rt)));
        rc = poll();
        if (rc) return rc;
        if (hp[G_OUT_DONE] != 0.0) converged = 1;
    }
    if (!converged) break;
    // The RECURSIVE residual of every column is below tol.  wd_solve_block promises the TRUE one: R = phihat - Ahat X in
    // fp64, per-column norms against tol (K_GL_INIT; they are what info.relres reports).  Columns that miss restart the
    // recurrence from the true residual, X kept.
    rc = gl_apply(c, dag, n, XE, tmp64, T);
    if (rc) return rc;
    GL_K((gl_true_resid<<<L.G, L.B, 0, st>>>(nv, phihat, T, S)));
    GL_K((gl_init<<<L.G, L.B, 0, st>>>(nv, n, rb, S, R, Rt, P, V)));
    rc = poll();
    if (rc) return rc;
    converged = hp[G_OUT_DONE] != 0.0 ? 1 : 0;
    if (converged || outer >= cap) break;
    }
#undef GL_K
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, XE, XO, PhiO, 1.0, c->kappa);
    if (rc) return rc;
    if (info) {
        info->n_rhs = n;
        info->outer_steps = flex ? calls : outer;      // flexible: preconditioner calls (the paper's count)
        info->inner_iters_total = flex ? (int)hp[G_ITERS] : outer;
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

// ================================================================================================================
// Block BiCGStab (PAPER.md:72 ref. [7], case C of Table 1), fp64, unpreconditioned, on the
// even/odd system:   R = R~ = P = Bhat
//     V = Ahat P;  (R~^dag V) alpha = R~^dag R;  S = R - V alpha;  T = Ahat S;  omega = <T,S>_F / <T,T>_F;
//     X += P alpha + omega S;  R = S - omega T;  (R~^dag V) beta = -R~^dag T;  P = R + (P - omega V) beta
// alpha, beta are n x n complex matrices; a block element (k, site) holds its n columns contiguously (RHS-minor layout),
// so the tall-skinny products are per-element n x n work with the Gram sums reduced over the lattice.
// ================================================================================================================
namespace {

enum { BL_MG = 0, BL_MR = 1, BL_MT = 2, BL_ALPHA = 3, BL_BETA = 4, BL_NMAT = 5 };
constexpr int BL_LD = 2 * WD_MAX_RHS * WD_MAX_RHS;   // doubles per matrix

// Every kernel of a Block BiCGStab iteration is a no-op once the recurrence has broken down or every column has converged:
// iterations enqueued between two polls of the host then leave X and R at the last good iterate (wd.h: X holds the best
// iterate on WD_ENOCONV).
__device__ __forceinline__ bool bl_frozen(const double* scal) { return scal[G_GL_BREAK] != 0.0 || scal[G_OUT_DONE] != 0.0; }

// MA[i][j] = sum_g conj(Rt[g,i]) A[g,j]   (and MB with B when B != null), written, not accumulated; one thread per
// (g, i, j), stride % n^2 == 0.  The sums are added in a fixed order (threads of one entry within a block in index
// order, then the block partials in block order by the last block to finish), so the result is the same run to run,
// like every other reduction of the library.  partials: gridDim.x * (B ? 4 : 2) * n * n doubles.
__global__ void bl_gram(long ng, int n, const double2* __restrict__ Rt, const double2* __restrict__ A, const double2* B, double* MA, double* MB,
                        const double* __restrict__ scal, double* partials, unsigned int* ticket) {
    if (bl_frozen(scal)) return;
    extern __shared__ double shg[];   // [4][blockDim.x]
    __shared__ bool is_last;
    const int nn = n * n, t = threadIdx.x, Bd = blockDim.x;
    const long total = ng * nn, stride = (long)gridDim.x * Bd;
    const long i0 = (long)blockIdx.x * Bd + t;
    const int ij = (int)(i0 % nn), i = ij / n, j = ij - i * n;
    double ar = 0.0, ai = 0.0, br = 0.0, bi = 0.0;
    for (long idx = i0; idx < total; idx += stride) {
        const long g = idx / nn;
        const double2 q = Rt[g * n + i], a = A[g * n + j];
        ar += q.x * a.x + q.y * a.y;
        ai += q.x * a.y - q.y * a.x;
        if (B) {
            const double2 b = B[g * n + j];
            br += q.x * b.x + q.y * b.y;
            bi += q.x * b.y - q.y * b.x;
        }
    }
    shg[t] = ar; shg[Bd + t] = ai; shg[2 * Bd + t] = br; shg[3 * Bd + t] = bi;
    __syncthreads();
    // item k = ((matrix m) * nn + entry) * 2 + (re, im): the layout of MA followed by MB
    const int items = (B ? 4 : 2) * nn;
    for (int k = t; k < items; k += Bd) {
        const int cpl = k & 1, e = k >> 1, m = e / nn, ent = e - m * nn;
        double sum = 0.0;
        for (int q = ent; q < Bd; q += nn) sum += shg[(2 * m + cpl) * Bd + q];
        partials[(size_t)blockIdx.x * items + k] = sum;
    }
    __threadfence();
    __syncthreads();
    if (t == 0) is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int k = t; k < items; k += Bd) {
        double sum = 0.0;
        for (unsigned g = 0; g < gridDim.x; ++g) sum += __ldcg(partials + (size_t)g * items + k);
        const int e = k >> 1, m = e / nn;
        (m ? MB : MA)[k - 2 * m * nn] = sum;
    }
    if (t == 0) *ticket = 0u;
}

// OUT = sign * MG^-1 RHS  (n x n complex, row-major, Gaussian elimination with partial pivoting; one thread).
// A pivot below 1e-13 of the largest entry of MG means the block has lost rank (a zero column, two equal columns, or
// the recurrence itself breaking down): OUT = 0 and the break flag is set, which freezes X and R (bl_frozen).
__global__ void bl_small_solve(int n, const double* __restrict__ MG, const double* __restrict__ RHS, double* OUT, double sign, double* scal) {
    if (bl_frozen(scal)) return;
    double2 a[WD_MAX_RHS][WD_MAX_RHS], b[WD_MAX_RHS][WD_MAX_RHS];
    double amax2 = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            a[i][j] = make_double2(MG[2 * (i * n + j)], MG[2 * (i * n + j) + 1]);
            b[i][j] = make_double2(sign * RHS[2 * (i * n + j)], sign * RHS[2 * (i * n + j) + 1]);
            const double m2 = a[i][j].x * a[i][j].x + a[i][j].y * a[i][j].y;
            if (m2 > amax2) amax2 = m2;
        }
    const double floor2 = 1e-26 * amax2;
    for (int k = 0; k < n; ++k) {
        int piv = k;
        double best = a[k][k].x * a[k][k].x + a[k][k].y * a[k][k].y;
        for (int i = k + 1; i < n; ++i) {
            const double m = a[i][k].x * a[i][k].x + a[i][k].y * a[i][k].y;
            if (m > best) { best = m; piv = i; }
        }
        if (!(best > floor2)) {   // also catches NaN
            for (int q = 0; q < 2 * n * n; ++q) OUT[q] = 0.0;
            scal[G_GL_BREAK] = 1.0;
            return;
        }
        if (piv != k)
            for (int j = 0; j < n; ++j) { double2 t = a[k][j]; a[k][j] = a[piv][j]; a[piv][j] = t; t = b[k][j]; b[k][j] = b[piv][j]; b[piv][j] = t; }
        const double2 inv = make_double2(a[k][k].x / best, -a[k][k].y / best);
        for (int i = k + 1; i < n; ++i) {
            const double2 f = make_double2(a[i][k].x * inv.x - a[i][k].y * inv.y, a[i][k].x * inv.y + a[i][k].y * inv.x);
            for (int j = k; j < n; ++j) { a[i][j].x -= f.x * a[k][j].x - f.y * a[k][j].y; a[i][j].y -= f.x * a[k][j].y + f.y * a[k][j].x; }
            for (int j = 0; j < n; ++j) { b[i][j].x -= f.x * b[k][j].x - f.y * b[k][j].y; b[i][j].y -= f.x * b[k][j].y + f.y * b[k][j].x; }
        }
    }
    for (int k = n - 1; k >= 0; --k) {
        const double d = a[k][k].x * a[k][k].x + a[k][k].y * a[k][k].y;
        const double2 inv = make_double2(a[k][k].x / d, -a[k][k].y / d);
        for (int j = 0; j < n; ++j) {
            double2 s = b[k][j];
            for (int m = k + 1; m < n; ++m) { s.x -= a[k][m].x * b[m][j].x - a[k][m].y * b[m][j].y; s.y -= a[k][m].x * b[m][j].y + a[k][m].y * b[m][j].x; }
            b[k][j] = make_double2(s.x * inv.x - s.y * inv.y, s.x * inv.y + s.y * inv.x);
        }
    }
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) { OUT[2 * (i * n + j)] = b[i][j].x; OUT[2 * (i * n + j) + 1] = b[i][j].y; }
}

// out[g,i] = base[g,i] + csign * sum_j (A[g,j] - w B[g,j]) M[j][i]   (B nullable: w ignored); thread = (g, i)
__global__ void bl_axpm(long nvec, int n, const double2* __restrict__ Base, const double2* __restrict__ A, const double2* B,
                        const double* __restrict__ scal, const double* __restrict__ M, double csign, double2* Out) {
    if (bl_frozen(scal)) return;
    extern __shared__ double shm[];   // M: [n][n][2]
    for (int k = threadIdx.x; k < 2 * n * n; k += blockDim.x) shm[k] = M[k];
    __syncthreads();
    const double wr = scal[G_GL_OMEGA_RE], wi = scal[G_GL_OMEGA_IM];
    const long stride = (long)gridDim.x * blockDim.x;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < nvec; idx += stride) {
        const long g = idx / n;
        const int i = (int)(idx - g * n);
        double2 acc = make_double2(0.0, 0.0);
        for (int j = 0; j < n; ++j) {
            double2 a = A[g * n + j];
            if (B) { const double2 wb = cmul2(wr, wi, B[g * n + j]); a.x -= wb.x; a.y -= wb.y; }
            const double mr = shm[2 * (j * n + i)], mi = shm[2 * (j * n + i) + 1];
            acc.x += a.x * mr - a.y * mi;
            acc.y += a.x * mi + a.y * mr;
        }
        const double2 b0 = Base[idx];
        Out[idx] = make_double2(b0.x + csign * acc.x, b0.y + csign * acc.y);
    }
}

// X += P alpha + omega S;  R = S - omega T;  |R_i|^2 -> per-column convergence
__global__ void bl_xr_update(long nvec, int n, RedBuf rb, double2* X, const double2* __restrict__ P, const double* __restrict__ ALPHA,
                             const double2* __restrict__ S, const double2* __restrict__ T, double2* R) {
    if (bl_frozen(rb.scal)) return;
    extern __shared__ double shm[];
    for (int k = threadIdx.x; k < 2 * n * n; k += blockDim.x) shm[k] = ALPHA[k];
    __syncthreads();
    const double wr = rb.scal[G_GL_OMEGA_RE], wi = rb.scal[G_GL_OMEGA_IM];
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < nvec; idx += stride) {
        const long g = idx / n;
        const int i = (int)(idx - g * n);
        double2 acc = make_double2(0.0, 0.0);
        for (int j = 0; j < n; ++j) {
            const double2 a = P[g * n + j];
            const double mr = shm[2 * (j * n + i)], mi = shm[2 * (j * n + i) + 1];
            acc.x += a.x * mr - a.y * mi;
            acc.y += a.x * mi + a.y * mr;
        }
        const double2 sv = S[idx], ws = cmul2(wr, wi, sv), wt = cmul2(wr, wi, T[idx]);
        double2 x = X[idx];
        x.x += acc.x + ws.x; x.y += acc.y + ws.y;
        X[idx] = x;
        const double2 r = make_double2(sv.x - wt.x, sv.y - wt.y);
        R[idx] = r;
        s[0] += r.x * r.x + r.y * r.y;
    }
    reduce_finalize<1, K_GL_S>(s, n, rb);
}

// R = R~ = P = B; per-column |B_i|^2 -> convergence flags
__global__ void bl_init(long nvec, int n, RedBuf rb, const double2* __restrict__ Bv, double2* R, double2* Rt, double2* P) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 b = Bv[i];
        R[i] = b; Rt[i] = b; P[i] = b;
        s[0] += b.x * b.x + b.y * b.y;
    }
    reduce_finalize<1, K_GL_INIT>(s, n, rb);
}

}  // namespace

int wd_solve_bl(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_iters, wd_solve_info* info) {
    const auto t_begin = std::chrono::steady_clock::now();
    cudaStream_t st = c->stream;
    const long Vh = c->Vh;
    const size_t hb64 = wd_half_bytes(c, WD_F64, n);
    const size_t sb64 = wd_align_up(wd_half_bytes(c, WD_F64, c->max_rhs));
    double2* phihat = (double2*)c->d_solver;
    double2* tmp64 = (double2*)(c->d_solver + sb64);
    double2* R = (double2*)(c->d_solver + 2 * sb64);
    double2 *Rt = gl_block(c, 0), *P = gl_block(c, 1), *V = gl_block(c, 2), *S = gl_block(c, 3), *T = gl_block(c, 4), *Pn = gl_block(c, 7);
    double* mats = c->d_partials + c->partial_doubles - (size_t)BL_NMAT * BL_LD;   // behind anything a reduction of this solver writes
    const char* PhiE = (const char*)Phi;
    const char* PhiO = PhiE + hb64;
    double2* XE = (double2*)X;
    char* XO = (char*)X + hb64;
    RedBuf rb{c->d_scal, c->d_partials, c->d_ticket};
    const long nv = 12 * Vh * n, ng = 12 * Vh;
    const GlLaunch L = gl_cfg(c, nv, n), Lf = gl_cfg(c, 2 * nv, n);
    const int nn = n * n;
    const int Bg = nn * (256 / nn > 0 ? 256 / nn : 1);
    // Gram kernel: its per-block partial sums (4 n^2 doubles a block) share d_partials with the matrices at its tail
    const size_t gram_room = (c->partial_doubles - (size_t)BL_NMAT * BL_LD) / (size_t)(4 * nn);
    const unsigned Gg = (unsigned)(gram_room < (size_t)c->n_sm * 4 ? gram_room : (size_t)c->n_sm * 4);
    const size_t shM = sizeof(double) * 2 * nn, shG = sizeof(double) * 4 * Bg;
    double* hp = c->h_pinned;
    int rc;
#define BL_K(call) { wd_prof_scope pr__(c, WD_PROF_BLAS); call; } WD_LAUNCH_CHECK(c)
    BL_K((gl_set_globals<<<1, 1, 0, st>>>(c->d_scal, tol * tol, 0.0)));
    BL_K((gl_norm2<<<Lf.G, Lf.B, 0, st>>>(2 * nv, n, rb, (const double2*)Phi)));
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 0, PhiO, phihat, PhiE, 1.0, c->kappa);
    if (rc) return rc;
    WD_CUDA_CHECK(c, cudaMemsetAsync(XE, 0, hb64, st));
    BL_K((bl_init<<<L.G, L.B, 0, st>>>(nv, n, rb, phihat, R, Rt, P)));
    WD_CUDA_CHECK(c, cudaMemsetAsync(mats, 0, sizeof(double) * BL_NMAT * BL_LD, st));   // alpha and beta too: nothing is ever read unset
    WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
    WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
    int converged = hp[G_OUT_DONE] != 0.0 ? 1 : 0, it = 0;
    const int poll_every = c->opt[WD_OPT_POLL_EVERY];
    for (;;) {
    while (!converged && it < max_iters) {
        ++it;
        rc = gl_apply(c, dag, n, P, tmp64, V);
        if (rc) return rc;
        BL_K((bl_gram<<<Gg, Bg, shG, st>>>(ng, n, Rt, V, R, mats + BL_MG * BL_LD, mats + BL_MR * BL_LD, c->d_scal, c->d_partials, c->d_ticket)));
        BL_K((bl_small_solve<<<1, 1, 0, st>>>(n, mats + BL_MG * BL_LD, mats + BL_MR * BL_LD, mats + BL_ALPHA * BL_LD, 1.0, c->d_scal)));
        BL_K((bl_axpm<<<L.G, L.B, shM, st>>>(nv, n, R, V, nullptr, c->d_scal, mats + BL_ALPHA * BL_LD, -1.0, S)));   // S = R - V alpha
        rc = gl_apply(c, dag, n, S, tmp64, T);
        if (rc) return rc;
        BL_K((gl_omega<<<L.G, L.B, 0, st>>>(nv, n, rb, T, S)));
        BL_K((bl_xr_update<<<L.G, L.B, shM, st>>>(nv, n, rb, XE, P, mats + BL_ALPHA * BL_LD, S, T, R)));
        BL_K((bl_gram<<<Gg, Bg, shG, st>>>(ng, n, Rt, T, nullptr, mats + BL_MT * BL_LD, nullptr, c->d_scal, c->d_partials, c->d_ticket)));
        BL_K((bl_small_solve<<<1, 1, 0, st>>>(n, mats + BL_MG * BL_LD, mats + BL_MT * BL_LD, mats + BL_BETA * BL_LD, -1.0, c->d_scal)));
        BL_K((bl_axpm<<<L.G, L.B, shM, st>>>(nv, n, R, P, V, c->d_scal, mats + BL_BETA * BL_LD, 1.0, Pn)));           // P = R + (P - omega V) beta
        { double2* t = P; P = Pn; Pn = t; }
        if (it % poll_every == 0 || it == max_iters) {
            WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
            WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
            if (hp[G_OUT_DONE] != 0.0) converged = 1;
            if (hp[G_GL_BREAK] != 0.0) break;
        }
    }
    if (!converged) break;
    // recursive residuals below tol: check the true residual and restart from it where it misses (as in wd_solve_gl)
    rc = gl_apply(c, dag, n, XE, tmp64, T);
    if (rc) return rc;
    BL_K((gl_true_resid<<<L.G, L.B, 0, st>>>(nv, phihat, T, S)));
    BL_K((bl_init<<<L.G, L.B, 0, st>>>(nv, n, rb, S, R, Rt, P)));
    WD_CUDA_CHECK(c, cudaMemcpyAsync(hp, c->d_scal, sizeof(double) * G_COUNT, cudaMemcpyDeviceToHost, st));
    WD_CUDA_CHECK(c, cudaStreamSynchronize(st));
    converged = hp[G_OUT_DONE] != 0.0 ? 1 : 0;
    if (converged || it >= max_iters) break;
    }
#undef BL_K
    // The block recurrence broke down (rank-deficient block: a zero column, two equal columns, or a true breakdown):
    // X and R are frozen at the last good iterate, and the caller (wd_solve_impl) finishes the solve on the default route.
    if (!converged && hp[G_GL_BREAK] != 0.0) return WD_BL_BREAKDOWN;
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, dag, n, 1, XE, XO, PhiO, 1.0, c->kappa);
    if (rc) return rc;
    if (info) {
        info->n_rhs = n;
        info->outer_steps = it;
        info->inner_iters_total = it;
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
