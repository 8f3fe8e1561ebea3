// wd_blas.cuh -- batched-per-RHS BLAS1 updates fused with their inner products (hot-path step a4)
// and the device-side scalar recurrences of BiCGStab (textbook BiCGStab per column; the schedule is DESIGN.md section 6).
//
// Thread mapping: a block has B = 32*n*m threads (m = ceil(8/n)), so B is a multiple of n and thread
// t always works on column r = t % n of the flat RHS-minor vector index.  Per-column sums go
// thread -> shared memory (transposed so one warp owns one column) -> warp shuffle -> one partial
// per block and column in global memory -> the LAST block to finish (atomic ticket) adds the
// partials in a fixed order and runs the scalar recurrence, so no scalar ever visits the host and
// the result does not depend on block scheduling.  All sums are accumulated in fp64.
#pragma once
#include "wd_internal.h"

namespace wdblas {

// ---- layout of the per-column scalar table (doubles, column stride WD_MAX_RHS) -------------------
enum {
    S_RHO_RE = 0, S_RHO_IM, S_ALPHA_RE, S_ALPHA_IM, S_OMEGA_RE, S_OMEGA_IM, S_BETA_RE, S_BETA_IM,
    S_RNORM2,     // recursive |r_i|^2 of the inner solver
    S_THR2,       // inner stopping threshold on |r_i|^2
    S_FLAG,       // 0 active, 1 converged (frozen), 2 breakdown (frozen)
    S_OUT_R2,     // outer true residual |R_i|^2 (even/odd system)
    S_PHI2,       // |phi_i|^2 over the full lattice
    S_SCALE,      // |R_i| used to normalise the inner right-hand side
    S_OUT_CONV,   // 1 if column met the outer tolerance
    S_ACTION,     // |x_i|^2 of wd_action (pseudo-fermion action per column)
    S_RHO_PREV_RE, S_RHO_PREV_IM,  // rho of the previous iteration (reliable updates: beta is recomputed after r is replaced)
    S_RMAX2,      // largest recursive |r_i|^2 since the last reliable update
    S_T0, S_T1, S_T2,  // per-column totals of the global (Frobenius) inner products of the blocked outer solvers
    S_GL_CONV,    // column met the tolerance (blocked outer solvers)
    S_ROWS
};
// global (not per-column) slots after the table
enum { G_DONE = S_ROWS * WD_MAX_RHS, G_ITERS, G_OUT_DONE, G_TOL2, G_INTOL2, G_DELTA2, G_UPDATES,
       G_GL_RHO_RE, G_GL_RHO_IM, G_GL_ALPHA_RE, G_GL_ALPHA_IM, G_GL_OMEGA_RE, G_GL_OMEGA_IM, G_GL_BETA_RE, G_GL_BETA_IM, G_GL_BREAK,
       G_COUNT };

__device__ __forceinline__ double& SC(double* scal, int row, int r) { return scal[row * WD_MAX_RHS + r]; }

enum Kind { K_SIGMA, K_OMEGA, K_RHO, K_PHI2, K_OUT_R2, K_INIT_RHO, K_ACTION,
            K_OMEGA_RHO, K_RNORM,                  // merged-update schedule of the fp32 solver (wd_solve.cu)
            K_RHO_REL, K_OUT_R2_REL, K_REPLACE,     // reliable-update solver (wd_solve_h16.cu)
            K_GL_INIT, K_GL_SIGMA, K_GL_S, K_GL_OMEGA, K_GL_RHO, K_PREC_PREP };   // blocked outer solvers (wd_solve_gl.cu)

struct RedBuf {
    double* scal;
    double* partials;
    unsigned int* ticket;
    // optional residual history (wd_set_residual_history): row k = after inner iteration k, WD_MAX_RHS doubles a row.
    // Aggregate initialisation with three members leaves it off.
    double* hist = nullptr;
    int hist_cap = 0;
};

template <typename T> struct V;
template <> struct V<float> { typedef float4 type; enum { NC = 2 }; };
template <> struct V<double> { typedef double2 type; enum { NC = 1 }; };

struct cd { double re, im; };
__device__ __forceinline__ cd cmul(cd a, cd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cd cdiv(cd a, cd b) {
    const double d = b.re * b.re + b.im * b.im;
    return {(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}

// ---- scalar recurrences, run by one thread per column in the last block ---------------------------
template <int KIND>
__device__ void finalize_column(double* scal, int r, const double* tot) {
    const bool frozen = SC(scal, S_FLAG, r) != 0.0;
    if (KIND == K_SIGMA) {  // tot = <rt, v>;  alpha = rho / sigma
        cd alpha = {0.0, 0.0};
        if (!frozen) {
            const cd sigma = {tot[0], tot[1]};
            if (sigma.re == 0.0 && sigma.im == 0.0) SC(scal, S_FLAG, r) = 2.0;
            else alpha = cdiv({SC(scal, S_RHO_RE, r), SC(scal, S_RHO_IM, r)}, sigma);
        }
        SC(scal, S_ALPHA_RE, r) = alpha.re;
        SC(scal, S_ALPHA_IM, r) = alpha.im;
    } else if (KIND == K_OMEGA) {  // tot = <t, s>, <t, t>;  omega = <t,s>/<t,t>
        cd omega = {0.0, 0.0};
        if (!frozen && tot[2] > 0.0) omega = {tot[0] / tot[2], tot[1] / tot[2]};
        SC(scal, S_OMEGA_RE, r) = omega.re;
        SC(scal, S_OMEGA_IM, r) = omega.im;
    } else if (KIND == K_OMEGA_RHO) {
        // tot = <t,s> (2), <t,t>, <rt,s> (2), <rt,t> (2): omega as above, and the NEXT rho without waiting for the new r,
        // rho' = <rt, s - omega t> = <rt,s> - omega <rt,t>, so that beta is known before the merged x, r, p update runs
        cd omega = {0.0, 0.0}, beta = {0.0, 0.0};
        if (!frozen && tot[2] > 0.0) omega = {tot[0] / tot[2], tot[1] / tot[2]};
        SC(scal, S_OMEGA_RE, r) = omega.re;
        SC(scal, S_OMEGA_IM, r) = omega.im;
        if (!frozen) {
            const cd wt = cmul(omega, {tot[5], tot[6]});
            const cd rho1 = {tot[3] - wt.re, tot[4] - wt.im};
            const cd rho = {SC(scal, S_RHO_RE, r), SC(scal, S_RHO_IM, r)};
            const cd alpha = {SC(scal, S_ALPHA_RE, r), SC(scal, S_ALPHA_IM, r)};
            if (!(rho1.re == rho1.re) || !(rho1.im == rho1.im) || (omega.re == 0.0 && omega.im == 0.0) ||
                (rho1.re == 0.0 && rho1.im == 0.0) || (rho.re == 0.0 && rho.im == 0.0)) {
                SC(scal, S_FLAG, r) = 2.0;  // breakdown or NaN: the merged update still forms x and r; the outer loop restarts
            } else {
                beta = cmul(cdiv(rho1, rho), cdiv(alpha, omega));
            }
            SC(scal, S_RHO_RE, r) = rho1.re; SC(scal, S_RHO_IM, r) = rho1.im;
        }
        SC(scal, S_BETA_RE, r) = beta.re; SC(scal, S_BETA_IM, r) = beta.im;
    } else if (KIND == K_RNORM) {  // tot = |r|^2 after the merged x, r, p update: convergence only
        if (frozen) return;
        SC(scal, S_RNORM2, r) = tot[0];
        if (tot[0] <= SC(scal, S_THR2, r)) SC(scal, S_FLAG, r) = 1.0;
        else if (!(tot[0] == tot[0])) SC(scal, S_FLAG, r) = 2.0;
    } else if (KIND == K_RHO || KIND == K_INIT_RHO) {  // tot = <rt, r>, |r|^2
        if (KIND == K_INIT_RHO) {
            SC(scal, S_RHO_RE, r) = tot[0]; SC(scal, S_RHO_IM, r) = tot[1];
            SC(scal, S_ALPHA_RE, r) = 1.0;  SC(scal, S_ALPHA_IM, r) = 0.0;
            SC(scal, S_OMEGA_RE, r) = 1.0;  SC(scal, S_OMEGA_IM, r) = 0.0;
            SC(scal, S_BETA_RE, r) = 0.0;   SC(scal, S_BETA_IM, r) = 0.0;
            SC(scal, S_RNORM2, r) = tot[2];
            SC(scal, S_RMAX2, r) = tot[2];
            // S_FLAG was set by the outer residual kernel (1 = column already converged)
            if (!frozen && !(tot[2] > 0.0)) SC(scal, S_FLAG, r) = 1.0;
            return;
        }
        if (frozen) {
            SC(scal, S_BETA_RE, r) = 0.0; SC(scal, S_BETA_IM, r) = 0.0;
            return;
        }
        SC(scal, S_RNORM2, r) = tot[2];
        const cd rho1 = {tot[0], tot[1]};
        const cd rho = {SC(scal, S_RHO_RE, r), SC(scal, S_RHO_IM, r)};
        const cd alpha = {SC(scal, S_ALPHA_RE, r), SC(scal, S_ALPHA_IM, r)};
        const cd omega = {SC(scal, S_OMEGA_RE, r), SC(scal, S_OMEGA_IM, r)};
        cd beta = {0.0, 0.0};
        if (tot[2] <= SC(scal, S_THR2, r)) {
            SC(scal, S_FLAG, r) = 1.0;
        } else if (!(tot[2] == tot[2]) || (omega.re == 0.0 && omega.im == 0.0) || (rho1.re == 0.0 && rho1.im == 0.0)) {
            SC(scal, S_FLAG, r) = 2.0;  // breakdown or NaN: freeze; the outer loop restarts from the true residual
        } else {
            beta = cmul(cdiv(rho1, rho), cdiv(alpha, omega));
        }
        SC(scal, S_RHO_RE, r) = rho1.re; SC(scal, S_RHO_IM, r) = rho1.im;
        SC(scal, S_BETA_RE, r) = beta.re; SC(scal, S_BETA_IM, r) = beta.im;
    } else if (KIND == K_RHO_REL) {  // tot = <rt, r>, |r|^2 after the x, r update of the reliable-update solver
        if (frozen) {
            SC(scal, S_BETA_RE, r) = 0.0; SC(scal, S_BETA_IM, r) = 0.0;
            return;
        }
        SC(scal, S_RNORM2, r) = tot[2];
        const cd rho1 = {tot[0], tot[1]};
        const cd rho = {SC(scal, S_RHO_RE, r), SC(scal, S_RHO_IM, r)};
        const cd alpha = {SC(scal, S_ALPHA_RE, r), SC(scal, S_ALPHA_IM, r)};
        const cd omega = {SC(scal, S_OMEGA_RE, r), SC(scal, S_OMEGA_IM, r)};
        cd beta = {0.0, 0.0};
        if (tot[2] <= SC(scal, S_THR2, r)) {
            SC(scal, S_FLAG, r) = 1.0;   // converged by the recursive residual: the next reliable update checks the true one
        } else if (!(tot[2] == tot[2]) || (omega.re == 0.0 && omega.im == 0.0) || (rho1.re == 0.0 && rho1.im == 0.0)) {
            SC(scal, S_FLAG, r) = 2.0;   // breakdown or NaN: frozen until the next reliable update restarts the column
        } else {
            beta = cmul(cdiv(rho1, rho), cdiv(alpha, omega));
        }
        SC(scal, S_RHO_PREV_RE, r) = rho.re; SC(scal, S_RHO_PREV_IM, r) = rho.im;
        SC(scal, S_RHO_RE, r) = rho1.re; SC(scal, S_RHO_IM, r) = rho1.im;
        SC(scal, S_BETA_RE, r) = beta.re; SC(scal, S_BETA_IM, r) = beta.im;
        if (tot[2] > SC(scal, S_RMAX2, r)) SC(scal, S_RMAX2, r) = tot[2];
    } else if (KIND == K_REPLACE) {  // tot = <rt, r'>, |r'|^2 with r' the true residual that replaced r
        SC(scal, S_RNORM2, r) = tot[2];
        SC(scal, S_RMAX2, r) = tot[2];
        if (frozen) return;            // converged columns (S_FLAG set by K_OUT_R2_REL) stay frozen
        const cd rho1 = {tot[0], tot[1]};
        const cd rho = {SC(scal, S_RHO_PREV_RE, r), SC(scal, S_RHO_PREV_IM, r)};
        const cd alpha = {SC(scal, S_ALPHA_RE, r), SC(scal, S_ALPHA_IM, r)};
        const cd omega = {SC(scal, S_OMEGA_RE, r), SC(scal, S_OMEGA_IM, r)};
        cd beta = {0.0, 0.0};
        const bool bad = (omega.re == 0.0 && omega.im == 0.0) || (rho.re == 0.0 && rho.im == 0.0) || (rho1.re == 0.0 && rho1.im == 0.0);
        if (!bad) beta = cmul(cdiv(rho1, rho), cdiv(alpha, omega));
        else { SC(scal, S_OMEGA_RE, r) = 1.0; SC(scal, S_OMEGA_IM, r) = 0.0; SC(scal, S_ALPHA_RE, r) = 1.0; SC(scal, S_ALPHA_IM, r) = 0.0; }
        // after a breakdown the column restarts: beta = 0 makes p = r'; (alpha, omega reset; v is multiplied by beta = 0)
        SC(scal, S_RHO_RE, r) = rho1.re; SC(scal, S_RHO_IM, r) = rho1.im;
        SC(scal, S_BETA_RE, r) = beta.re; SC(scal, S_BETA_IM, r) = beta.im;
    } else if (KIND == K_OUT_R2_REL) {  // tot = |R_i|^2, the TRUE fp64 residual of the even/odd system
        SC(scal, S_OUT_R2, r) = tot[0];
        const double phi2 = SC(scal, S_PHI2, r);
        const double tol2 = scal[G_TOL2];
        const bool conv = tot[0] <= tol2 * phi2;
        SC(scal, S_OUT_CONV, r) = conv ? 1.0 : 0.0;
        SC(scal, S_FLAG, r) = conv ? 1.0 : 0.0;   // a column frozen on its recursive residual or a breakdown goes on if not converged
        if (scal[G_UPDATES] == 0.0) {             // first call: the normalisation of the low-precision system is fixed here
            SC(scal, S_SCALE, r) = sqrt(tot[0]);
            // recursive target: half of what the tolerance needs, in units of the scale
            SC(scal, S_THR2, r) = tot[0] > 0.0 ? 0.25 * tol2 * phi2 / tot[0] : 0.0;
        }
    } else if (KIND == K_GL_INIT || KIND == K_GL_S || KIND == K_GL_RHO) {
        // per-column part of a global inner product; the residual norm of the column is tot[0] (INIT, S) or tot[2] (RHO)
        const double r2 = KIND == K_GL_RHO ? tot[2] : tot[0];
        SC(scal, S_T0, r) = tot[0];
        if (KIND == K_GL_RHO) { SC(scal, S_T1, r) = tot[1]; SC(scal, S_T2, r) = tot[2]; }
        SC(scal, S_OUT_R2, r) = r2;
        SC(scal, S_GL_CONV, r) = r2 <= scal[G_TOL2] * SC(scal, S_PHI2, r) ? 1.0 : 0.0;
    } else if (KIND == K_GL_SIGMA) {
        SC(scal, S_T0, r) = tot[0]; SC(scal, S_T1, r) = tot[1];
    } else if (KIND == K_GL_OMEGA) {
        SC(scal, S_T0, r) = tot[0]; SC(scal, S_T1, r) = tot[1]; SC(scal, S_T2, r) = tot[2];
    } else if (KIND == K_PREC_PREP) {  // tot = |in_i|^2: the inner solver works on in_i / |in_i|
        SC(scal, S_SCALE, r) = sqrt(tot[0]);
        SC(scal, S_FLAG, r) = tot[0] > 0.0 ? 0.0 : 1.0;
        SC(scal, S_THR2, r) = scal[G_INTOL2];
        SC(scal, S_OUT_CONV, r) = 0.0;
    } else if (KIND == K_PHI2) {
        SC(scal, S_PHI2, r) = tot[0];
    } else if (KIND == K_ACTION) {
        SC(scal, S_ACTION, r) = tot[0];
    } else if (KIND == K_OUT_R2) {  // tot = |R_i|^2 of the fp64 even/odd system
        SC(scal, S_OUT_R2, r) = tot[0];
        const double phi2 = SC(scal, S_PHI2, r);
        const double tol2 = scal[G_TOL2];
        const bool conv = tot[0] <= tol2 * phi2;
        SC(scal, S_OUT_CONV, r) = conv ? 1.0 : 0.0;
        SC(scal, S_SCALE, r) = sqrt(tot[0]);
        SC(scal, S_FLAG, r) = conv ? 1.0 : 0.0;
        // inner target: the asked reduction, but never far below what the outer tolerance needs
        double thr2 = scal[G_INTOL2];
        if (tot[0] > 0.0) thr2 = fmax(thr2, 0.25 * tol2 * phi2 / tot[0]);
        SC(scal, S_THR2, r) = thr2;  // inner rhs is normalised to |b_i| = 1
    }
}

template <int KIND>
__device__ void finalize_global(double* scal, int n) {
    if (KIND == K_RHO || KIND == K_INIT_RHO || KIND == K_RNORM) {
        bool all = true;
        for (int r = 0; r < n; ++r) all = all && (SC(scal, S_FLAG, r) != 0.0);
        scal[G_DONE] = all ? 1.0 : 0.0;
        if (KIND != K_INIT_RHO) scal[G_ITERS] += 1.0;
    } else if (KIND == K_OUT_R2) {
        bool all = true;
        for (int r = 0; r < n; ++r) all = all && (SC(scal, S_OUT_CONV, r) != 0.0);
        scal[G_OUT_DONE] = all ? 1.0 : 0.0;
    } else if (KIND == K_RHO_REL) {
        // the iteration kernels turn into no-ops when every column is frozen OR a column asks for a reliable update
        // (its recursive residual fell below delta times the largest one since the last update)
        bool all = true, rel = false;
        for (int r = 0; r < n; ++r) {
            const bool fr = SC(scal, S_FLAG, r) != 0.0;
            all = all && fr;
            rel = rel || (!fr && SC(scal, S_RNORM2, r) < scal[G_DELTA2] * SC(scal, S_RMAX2, r));
        }
        scal[G_DONE] = (all || rel) ? 1.0 : 0.0;
        scal[G_ITERS] += 1.0;
    } else if (KIND == K_OUT_R2_REL) {
        bool all = true;
        for (int r = 0; r < n; ++r) all = all && (SC(scal, S_OUT_CONV, r) != 0.0);
        scal[G_OUT_DONE] = all ? 1.0 : 0.0;
        scal[G_UPDATES] += 1.0;
    } else if (KIND == K_REPLACE) {
        bool all = true;
        for (int r = 0; r < n; ++r) all = all && (SC(scal, S_FLAG, r) != 0.0);
        scal[G_DONE] = all ? 1.0 : 0.0;
    } else if (KIND == K_GL_INIT || KIND == K_GL_S || KIND == K_GL_RHO || KIND == K_GL_SIGMA || KIND == K_GL_OMEGA) {
        // Frobenius inner products = sums over the columns (PAPER.md:72 Gl-BiCGStab, ref. [6])
        double t0 = 0.0, t1 = 0.0, t2 = 0.0;
        bool all = true;
        for (int r = 0; r < n; ++r) {
            t0 += SC(scal, S_T0, r); t1 += SC(scal, S_T1, r); t2 += SC(scal, S_T2, r);
            all = all && (SC(scal, S_GL_CONV, r) != 0.0);
        }
        if (KIND == K_GL_INIT) {          // rho = <R~, R>_F with R~ = R
            scal[G_GL_RHO_RE] = t0; scal[G_GL_RHO_IM] = 0.0;
            scal[G_GL_ALPHA_RE] = 1.0; scal[G_GL_ALPHA_IM] = 0.0; scal[G_GL_OMEGA_RE] = 1.0; scal[G_GL_OMEGA_IM] = 0.0;
            scal[G_GL_BETA_RE] = 0.0; scal[G_GL_BETA_IM] = 0.0; scal[G_GL_BREAK] = 0.0;
            scal[G_OUT_DONE] = all ? 1.0 : 0.0;
        } else if (KIND == K_GL_SIGMA) {  // alpha = rho / <R~, V>_F
            const cd sigma = {t0, t1};
            cd alpha = {0.0, 0.0};
            if (sigma.re == 0.0 && sigma.im == 0.0) scal[G_GL_BREAK] = 1.0;
            else alpha = cdiv({scal[G_GL_RHO_RE], scal[G_GL_RHO_IM]}, sigma);
            scal[G_GL_ALPHA_RE] = alpha.re; scal[G_GL_ALPHA_IM] = alpha.im;
        } else if (KIND == K_GL_S) {
            scal[G_OUT_DONE] = all ? 1.0 : 0.0;
        } else if (KIND == K_GL_OMEGA) {  // omega = <T, S>_F / <T, T>_F
            cd omega = {0.0, 0.0};
            if (t2 > 0.0) omega = {t0 / t2, t1 / t2};
            else scal[G_GL_BREAK] = 1.0;
            scal[G_GL_OMEGA_RE] = omega.re; scal[G_GL_OMEGA_IM] = omega.im;
        } else {                          // K_GL_RHO: rho' = <R~, R>_F, beta = (rho'/rho)(alpha/omega)
            const cd rho1 = {t0, t1}, rho = {scal[G_GL_RHO_RE], scal[G_GL_RHO_IM]};
            const cd alpha = {scal[G_GL_ALPHA_RE], scal[G_GL_ALPHA_IM]}, omega = {scal[G_GL_OMEGA_RE], scal[G_GL_OMEGA_IM]};
            cd beta = {0.0, 0.0};
            if ((rho.re == 0.0 && rho.im == 0.0) || (omega.re == 0.0 && omega.im == 0.0)) scal[G_GL_BREAK] = 1.0;
            else beta = cmul(cdiv(rho1, rho), cdiv(alpha, omega));
            scal[G_GL_RHO_RE] = rho1.re; scal[G_GL_RHO_IM] = rho1.im;
            scal[G_GL_BETA_RE] = beta.re; scal[G_GL_BETA_IM] = beta.im;
            scal[G_OUT_DONE] = all ? 1.0 : 0.0;
        }
    }
}

// Block + grid reduction of K per-thread fp64 sums for column r = threadIdx.x % n, then finalize.
// Requires blockDim.x % n == 0, blockDim.x / 32 >= n, K * blockDim.x <= 2048.  Partials are stored
// item-major ([column * K + k][block]) so that the last block reads them coalesced; it adds them in an
// order fixed by (gridDim, blockDim) alone, so results do not depend on block scheduling.
template <int K, int KIND>
__device__ void reduce_finalize(double (&v)[K], int n, RedBuf rb) {
    __shared__ double sh[4 * 512];
    __shared__ bool is_last;
    const int B = blockDim.x, t = threadIdx.x;
    const int per = B / n;  // threads per column
    const int r = t % n, q = t / n;
#pragma unroll
    for (int k = 0; k < K; ++k) sh[k * B + r * per + q] = v[k];
    __syncthreads();
    const int warp = t >> 5, lane = t & 31;
    const int nwarps = B >> 5;
    const unsigned grid = gridDim.x;
    if (warp < n) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            double s = 0.0;
            for (int j = lane; j < per; j += 32) s += sh[k * B + warp * per + j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) rb.partials[(size_t)(warp * K + k) * grid + blockIdx.x] = s;
        }
    }
    __threadfence();
    __syncthreads();
    if (t == 0) is_last = (atomicAdd(rb.ticket, 1u) == grid - 1);
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // last block: every thread adds a strided slice of each item's partials, then warps, then thread `item`
    const int items = n * K;  // <= 48
    for (int item = 0; item < items; ++item) {
        const double* p = rb.partials + (size_t)item * grid;
        double s = 0.0;
        for (unsigned g = t; g < grid; g += B) s += __ldcg(p + g);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) sh[item * 32 + warp] = s;
    }
    __syncthreads();
    if (t < items) {
        double s = 0.0;
        for (int w = 0; w < nwarps; ++w) s += sh[t * 32 + w];
        sh[1536 + t] = s;
    }
    __syncthreads();
    if (t < n) finalize_column<KIND>(rb.scal, t, &sh[1536 + t * K]);
    // the kernels that close a BiCGStab iteration (they own the recursive |r_i|^2) append a row to the residual history:
    // |r_i| of the normalised low-precision system x its scale / |phi_i| = an estimate of |phi - A x| / |phi| per column
    if ((KIND == K_RHO || KIND == K_RNORM || KIND == K_RHO_REL) && rb.hist != nullptr && t < n) {
        const int it = (int)rb.scal[G_ITERS];   // iterations finished before this one, since the solve began
        if (it < rb.hist_cap) {
            const double phi2 = SC(rb.scal, S_PHI2, t);
            rb.hist[(size_t)it * WD_MAX_RHS + t] = phi2 > 0.0 ? sqrt(SC(rb.scal, S_RNORM2, t) / phi2) * SC(rb.scal, S_SCALE, t) : 0.0;
        }
    }
    __syncthreads();
    if (t == 0) {
        finalize_global<KIND>(rb.scal, n);
        *rb.ticket = 0u;
    }
}

// Two-kernel form for reducing kernels with very many blocks (the hop with fused inner products):
// block_partials() is the first half of reduce_finalize (no ticket); finalize_partials_kernel, launched
// right after with one block per (column, value) item, adds that item's partials in a fixed order, and
// the last of those blocks runs the scalar recurrences.  `totals` is n * K doubles of scratch.
template <int K>
__device__ void block_partials(double (&v)[K], int n, RedBuf rb) {
    __shared__ double sh[3 * 512];  // K * blockDim.x <= 1536; blockDim.x a multiple of 32 and of n
    const int B = blockDim.x, t = threadIdx.x;
    const int per = B / n;
    const int r = t % n, q = t / n;
#pragma unroll
    for (int k = 0; k < K; ++k) sh[k * B + r * per + q] = v[k];
    __syncthreads();
    const int warp = t >> 5, lane = t & 31, nwarps = B >> 5;
    for (int col = warp; col < n; col += nwarps) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            double s = 0.0;
            for (int j = lane; j < per; j += 32) s += sh[k * B + col * per + j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) rb.partials[(size_t)(col * K + k) * gridDim.x + blockIdx.x] = s;
        }
    }
}

template <int K, int KIND>
__global__ void __launch_bounds__(256) finalize_partials_kernel(int n, unsigned nblocks, RedBuf rb, double* totals) {
    if (rb.scal[G_DONE] != 0.0) return;
    __shared__ double shw[8];
    __shared__ bool is_last;
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
    const double* p = rb.partials + (size_t)blockIdx.x * nblocks;
    double s = 0.0;
    for (unsigned g = t; g < nblocks; g += 256) s += p[g];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) shw[warp] = s;
    __syncthreads();
    if (t == 0) {
        double tot = 0.0;
        for (int w = 0; w < 8; ++w) tot += shw[w];
        totals[blockIdx.x] = tot;
        __threadfence();
        is_last = (atomicAdd(rb.ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (t < n) {
        double tot[K];
#pragma unroll
        for (int k = 0; k < K; ++k) tot[k] = __ldcg(totals + t * K + k);
        finalize_column<KIND>(rb.scal, t, tot);
    }
    __syncthreads();
    if (t == 0) {
        finalize_global<KIND>(rb.scal, n);
        *rb.ticket = 0u;
    }
}

}  // namespace wdblas
