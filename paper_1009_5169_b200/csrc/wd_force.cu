// wd_force.cu -- fermion force accumulation (hot-path step a8; Algorithm 2 lines 4-6, PAPER.md:56-58,
// eq. 2.3; the functional f[x,y] is DESIGN.md reading R9):
//
//   W_mu(s)  = sum_i sum_spin  x_i(s+mu) (x) ((1-gamma_mu) y_i(s))^dag + ((1+gamma_mu) y_i(s+mu)) (x) x_i(s)^dag
//   F_mu(s) += 2 kappa TA[ U_mu(s) W_mu(s) ],   TA(M) = (M - M^dag)/2 - tr(M - M^dag)/6.
//
// Because P = 1 -+ gamma_mu satisfies P = P^dag = P^2/2, sum_spin a (x) (P b)^dag equals
// sum_{j=0,1} h(a)_j (x) h(b)_j^dag with h the half-spinor projection of the hop kernel, so each term
// costs 2 colour outer products instead of 4.
//
// One thread owns one (site, rhs) pair, rhs fastest (the same coalesced 128-bit loads as the hop);
// it forms its column's contribution to W for the four forward links of its site.  The sum over
// the n columns of a site goes through shared memory, then one thread per (site, mu) does U*W, TA
// and the read-modify-write of F.
#include "wd_su3.cuh"

using namespace wdk;

namespace {

struct ForceArgs {
    const double2* X;   // native full-lattice blocks
    const double2* Y;
    const double* U;    // native fp64 18-real links
    const int32_t* nbr; // [2][Vh][8]
    const int32_t* site_of;
    double* F;          // canonical
    long V, Vh;
    uint32_t RB, lg;    // native layout blocks (wd_internal.h); neighbour indices are packed (block << lg) | offset
    int n;
    int spb;            // sites per block
    double coef;        // 2 kappa
};

template <int MU>
__device__ __forceinline__ void force_dir(const ForceArgs& A, int p, long nb, int r, const cx<double> (&x0)[12],
                                          const cx<double> (&y0)[12], double* w /* [18] */) {
    const long stride = A.Vh * A.n;
    const long nbb = (long)((uint32_t)nb >> A.lg), nbo = (long)((uint32_t)nb & ((1u << A.lg) - 1u));
    const long rbn = (long)A.RB * A.n;
    const double2* Xn = A.X + (long)(1 - p) * 12 * stride + nbb * 12 * rbn;
    const double2* Yn = A.Y + (long)(1 - p) * 12 * stride + nbb * 12 * rbn;
    cx<double> x1[12], y1[12], a[6], b[6], c[6], d[6];
    load_spinor(Xn, rbn, nbo * A.n + r, x1);
    load_spinor(Yn, rbn, nbo * A.n + r, y1);
    project<MU, 1>(x1, a);   // (1 - gamma) x(s+mu)
    project<MU, 1>(y0, b);   // (1 - gamma) y(s)
    project<MU, -1>(y1, c);  // (1 + gamma) y(s+mu)
    project<MU, -1>(x0, d);  // (1 + gamma) x(s)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            double re = 0.0, im = 0.0;
#pragma unroll
            for (int s = 0; s < 2; ++s) {  // a_i conj(b_j) + c_i conj(d_j)
                const cx<double> ai = a[3 * s + i], bj = b[3 * s + j], ci = c[3 * s + i], dj = d[3 * s + j];
                re += ai.re * bj.re + ai.im * bj.im + ci.re * dj.re + ci.im * dj.im;
                im += ai.im * bj.re - ai.re * bj.im + ci.im * dj.re - ci.re * dj.im;
            }
            w[2 * (3 * i + j)] = re;
            w[2 * (3 * i + j) + 1] = im;
        }
}

__global__ void force_kernel(const ForceArgs A) {
    extern __shared__ double sh[];  // [4][18][spb*n]: component-major, so that the threads of a warp write consecutive words
    const int n = A.n, spb = A.spb;
    const int t = threadIdx.x;
    const int ls = t / n, r = t - ls * n;   // local site, column
    // Blocks alternate between the parities over the SAME run of site indices (block 2k: even sites k*spb.., block
    // 2k+1: the odd sites with those indices, their x-neighbours), so that what one parity reads as its own sites the
    // other reads as forward neighbours at about the same time, out of L2.  With all even blocks first and all odd
    // blocks after them every X, Y element came from DRAM twice (ncu r03: 1.79 GB read for 1.02 GB of input).
    const int p = (int)(blockIdx.x & 1u);
    const long h = (long)(blockIdx.x >> 1) * spb + ls;
    const long gsite = (long)p * A.Vh + h;           // index into [2][Vh]
    const bool active = t < spb * n && h < A.Vh;
    const long stride = A.Vh * n;
    if (active) {
        const int4 n0 = __ldg(reinterpret_cast<const int4*>(A.nbr + gsite * WD_NDIR));
        const int4 n1 = __ldg(reinterpret_cast<const int4*>(A.nbr + gsite * WD_NDIR) + 1);
        const int items = spb * n;
        double* w = sh + t;               // element (mu, k) of this thread's item at w[(mu * 18 + k) * items]
        if ((uint32_t)n0.x & WD_SITE_FROZEN) {  // SF t=0: x(s) = y(s) = 0, so W = 0
#pragma unroll
            for (int mu = 0; mu < 4; ++mu)
#pragma unroll
                for (int k = 0; k < 18; ++k) w[(mu * 18 + k) * items] = 0.0;
        } else {
            cx<double> x0[12], y0[12];
            const long hb = h / A.RB, ho = h - hb * A.RB, rbn = (long)A.RB * n;
            load_spinor(A.X + (long)p * 12 * stride + hb * 12 * rbn, rbn, ho * n + r, x0);
            load_spinor(A.Y + (long)p * 12 * stride + hb * 12 * rbn, rbn, ho * n + r, y0);
            double wl[18];
            force_dir<0>(A, p, n0.x, r, x0, y0, wl);
#pragma unroll
            for (int k = 0; k < 18; ++k) w[(0 * 18 + k) * items] = wl[k];
            force_dir<1>(A, p, n0.z, r, x0, y0, wl);
#pragma unroll
            for (int k = 0; k < 18; ++k) w[(1 * 18 + k) * items] = wl[k];
            force_dir<2>(A, p, n1.x, r, x0, y0, wl);
#pragma unroll
            for (int k = 0; k < 18; ++k) w[(2 * 18 + k) * items] = wl[k];
            force_dir<3>(A, p, n1.z, r, x0, y0, wl);
#pragma unroll
            for (int k = 0; k < 18; ++k) w[(3 * 18 + k) * items] = wl[k];
        }
    }
    __syncthreads();
    // one thread per (local site, mu): sum the n columns, then U*W, TA, F +=
    if (t < spb * 4) {
        const int ls2 = t >> 2, mu = t & 3;
        const int p2 = p;
        const long h2 = (long)(blockIdx.x >> 1) * spb + ls2;
        const long g2 = (long)p2 * A.Vh + h2;
        if (h2 < A.Vh) {
            const int items = spb * n;
            const double* w = sh + (long)mu * 18 * items + (long)ls2 * n;
            cx<double> W[9];
#pragma unroll
            for (int k = 0; k < 9; ++k) { W[k].re = 0.0; W[k].im = 0.0; }
            for (int rr = 0; rr < n; ++rr)
#pragma unroll
                for (int k = 0; k < 9; ++k) { W[k].re += w[(2 * k) * items + rr]; W[k].im += w[(2 * k + 1) * items + rr]; }
            cx<double> u[9], M[9];
            const long hb2 = h2 / A.RB;
            load_link<18>(A.U + (long)(mu * 2 + p2) * 18 * A.Vh + hb2 * 18 * A.RB, (long)A.RB, h2 - hb2 * A.RB, u);
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    double re = 0.0, im = 0.0;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        re += u[3 * i + k].re * W[3 * k + j].re - u[3 * i + k].im * W[3 * k + j].im;
                        im += u[3 * i + k].re * W[3 * k + j].im + u[3 * i + k].im * W[3 * k + j].re;
                    }
                    M[3 * i + j].re = re;
                    M[3 * i + j].im = im;
                }
            // tr(M - M^dag) = 2 i Im tr M
            const double tri = 2.0 * (M[0].im + M[4].im + M[8].im);
            double* f = A.F + ((long)mu * A.V + A.site_of[g2]) * 18;
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    double re = 0.5 * (M[3 * i + j].re - M[3 * j + i].re);
                    double im = 0.5 * (M[3 * i + j].im + M[3 * j + i].im);
                    if (i == j) im -= tri / 6.0;
                    f[2 * (3 * i + j)] += A.coef * re;
                    f[2 * (3 * i + j) + 1] += A.coef * im;
                }
        }
    }
}

}  // namespace

int wd_force_impl(wd_ctx* c, int n, const double* X, const double* Y, double* F) {
    ForceArgs A;
    A.X = (const double2*)X;
    A.Y = (const double2*)Y;
    A.U = c->d_U64[0];
    A.nbr = c->d_nbr;
    A.site_of = c->d_site_of;
    A.F = F;
    A.V = c->V;
    A.Vh = c->Vh;
    A.RB = c->RB;
    A.lg = c->rb_lg;
    A.n = n;
    // about 128 threads (255 registers each: 256 threads is all an SM holds); stage 2 needs 4 * spb of them
    A.spb = 128 / n < 1 ? 1 : (128 / n > 32 ? 32 : 128 / n);
    int B = A.spb * n;
    if (B < 4 * A.spb) B = 4 * A.spb;
    B = (B + 31) / 32 * 32;
    A.coef = 2.0 * c->kappa;
    const size_t smem = sizeof(double) * 4 * (size_t)A.spb * n * 18;
    WD_CUDA_CHECK(c, wd_ensure_smem_attr(c, (const void*)force_kernel, 160 * 1024));
    const unsigned G = 2u * (unsigned)((c->Vh + A.spb - 1) / A.spb);   // (run of spb site indices) x (parity)
    wd_prof_scope prof(c, WD_PROF_FORCE);
    force_kernel<<<G, B, smem, c->stream>>>(A);
    WD_LAUNCH_CHECK(c);
    return WD_OK;
}
