// wd_md.cu -- the steps either side of the blocked solve in a molecular-dynamics step:
//   pseudo-fermion refresh  phi_i = D eta_i                      (eq. 2.1-2.2: S = sum_i |D^-1 phi_i|^2)
//   action                  S_i = |x_i|^2, x_i = D^-1 phi_i      (for the Metropolis test)
//   the whole of Algorithm 2 on device-resident fields, in two variants:
//     WD_ACTION_FULL  eq. 2.2 on the full operator: X = D^-1 Phi, Y = D^dag^-1 X
//     WD_ACTION_EO    the pseudo-fermions live on the even sites and the action is written on the even/odd-
//                     preconditioned operator Dhat = 1 - kappa^2 H_eo H_oe: S = sum_i |Dhat^-1 phi_i|^2.
//                     Because D (x_e, kappa H_oe x_e) = (Dhat x_e, 0), this is X = D^-1 (P_e Phi), Y = D^dag^-1 (P_e X) with
//                     the SAME force functional f[x, y] (reading R16; pinned in tests/test_oracle_pins.py by
//                     finite differences of the dense Schur-complement action).
// Every step is one of the library's kernels; this file only sequences them.
#include "wd_blas.cuh"

using namespace wdblas;

namespace {

// per-column sum of squares of a native fp64 block (full lattice or one parity half)
__global__ void action_kernel(long nvec, int n, RedBuf rb, const double2* __restrict__ A) {
    const long stride = (long)gridDim.x * blockDim.x;
    double s[1] = {0.0};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const double2 a = A[i];
        s[0] += a.x * a.x + a.y * a.y;
    }
    reduce_finalize<1, K_ACTION>(s, n, rb);
}

void blas_shape(const wd_ctx* c, long nvec, int n, int* B, unsigned* G) {
    const int m = (8 + n - 1) / n;
    *B = 32 * n * m;
    long g = (nvec + *B - 1) / *B;
    const long cap = (long)c->n_sm * 4;
    *G = (unsigned)(g < cap ? (g < 1 ? 1 : g) : cap);
}

}  // namespace

int wd_action_impl(wd_ctx* c, int n, int parity_sel, const double* X, double* S_host) {
    const long half = 12 * c->Vh * n;   // double2 elements of one parity half
    const double2* p = (const double2*)X + (parity_sel == WD_PARITY_ODD ? half : 0);
    const long nvec = parity_sel == WD_PARITY_BOTH ? 2 * half : half;
    int B; unsigned G;
    blas_shape(c, nvec, n, &B, &G);
    RedBuf rb{c->d_scal, c->d_partials, c->d_ticket};
    { wd_prof_scope pr__(c, WD_PROF_BLAS); action_kernel<<<G, B, 0, c->stream>>>(nvec, n, rb, p); }
    WD_LAUNCH_CHECK(c);
    WD_CUDA_CHECK(c, cudaMemcpyAsync(c->h_pinned + 512, c->d_scal + S_ACTION * WD_MAX_RHS, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    WD_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    for (int r = 0; r < n; ++r) S_host[r] = c->h_pinned[512 + r];
    return WD_OK;
}

// native = P_parity native: the other parity's half is zeroed (native blocks are [parity 0 half][parity 1 half])
int wd_project_parity_impl(wd_ctx* c, int prec, int n, int parity, void* native) {
    const size_t hb = wd_half_bytes(c, prec, n);
    WD_CUDA_CHECK(c, cudaMemsetAsync((char*)native + (size_t)(1 - parity) * hb, 0, hb, c->stream));
    return WD_OK;
}

int wd_refresh_impl(wd_ctx* c, int variant, int n, const double* eta, double* phi) {
    const size_t hb = wd_half_bytes(c, WD_F64, n);
    if (variant == WD_ACTION_FULL) {
        // phi = D eta: two fp64 hops with the diagonal term fused
        for (int p = 0; p < 2; ++p) {
            const int rc = wd_hop_launch(c, WD_F64, WD_LINK18, 0, n, p, (const char*)eta + (1 - p) * hb, (char*)phi + p * hb,
                                         (const char*)eta + p * hb, 1.0, -c->kappa);
            if (rc) return rc;
        }
        return WD_OK;
    }
    // phi_e = Dhat eta_e = eta_e - kappa^2 H_eo H_oe eta_e, phi_o = 0 (the odd half of phi is scratch for H_oe eta_e first)
    int rc = wd_hop_launch(c, WD_F64, WD_LINK18, 0, n, 1, eta, (char*)phi + hb, nullptr, 0.0, 1.0);
    if (rc) return rc;
    rc = wd_hop_launch(c, WD_F64, WD_LINK18, 0, n, 0, (char*)phi + hb, phi, eta, 1.0, -c->kappa * c->kappa);
    if (rc) return rc;
    WD_CUDA_CHECK(c, cudaMemsetAsync((char*)phi + hb, 0, hb, c->stream));
    return WD_OK;
}

// Algorithm 2 on device-resident native fields.  tmp: a native fp64 full-lattice block of scratch (EO variant only).
int wd_md_force_impl(wd_ctx* c, int variant, int n, const double* Phi, double* X, double* Y, double* F, double* S_host,
                     double* tmp, double tol, int max_outer, int max_inner, double inner_tol, int recon,
                     wd_solve_info* info2) {
    const size_t hb = wd_half_bytes(c, WD_F64, n);
    const double* rhs1 = Phi;
    if (variant == WD_ACTION_EO) {   // right-hand side P_e Phi
        WD_CUDA_CHECK(c, cudaMemcpyAsync(tmp, Phi, hb, cudaMemcpyDeviceToDevice, c->stream));
        WD_CUDA_CHECK(c, cudaMemsetAsync((char*)tmp + hb, 0, hb, c->stream));
        rhs1 = tmp;
    }
    const int rc1 = wd_solve_impl(c, 0, n, rhs1, X, tol, max_outer, max_inner, inner_tol, recon, info2 ? &info2[0] : nullptr);
    if (rc1 != WD_OK && rc1 != WD_ENOCONV) return rc1;
    const double* rhs2 = X;
    if (variant == WD_ACTION_EO) {   // right-hand side P_e X
        WD_CUDA_CHECK(c, cudaMemcpyAsync(tmp, X, hb, cudaMemcpyDeviceToDevice, c->stream));
        WD_CUDA_CHECK(c, cudaMemsetAsync((char*)tmp + hb, 0, hb, c->stream));
        rhs2 = tmp;
    }
    const int rc2 = wd_solve_impl(c, 1, n, rhs2, Y, tol, max_outer, max_inner, inner_tol, recon, info2 ? &info2[1] : nullptr);
    if (rc2 != WD_OK && rc2 != WD_ENOCONV) return rc2;
    if (S_host) {
        const int rc = wd_action_impl(c, n, variant == WD_ACTION_EO ? WD_PARITY_EVEN : WD_PARITY_BOTH, X, S_host);
        if (rc) return rc;
    }
    const int rc = wd_force_impl(c, n, X, Y, F);
    if (rc) return rc;
    return (rc1 == WD_OK && rc2 == WD_OK) ? WD_OK : WD_ENOCONV;
}
