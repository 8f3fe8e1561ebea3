// wd_hop.cu -- the multi-RHS even/odd Wilson hopping kernel (hot-path step a2; PAPER.md:80-84,
// "single-precision coefficient matrix D on the GPUs is also even/odd preconditioned").
//
//   (H psi)(x) = sum_mu (1 -+ gamma_mu) U_mu(x) psi(x+mu) + (1 +- gamma_mu) U_mu(x-mu)^dag psi(x-mu)
//   (upper sign D, lower sign D^dag) on ONE output parity, for all n_rhs columns in one launch,
//   optionally with the fused epilogue out = a*in2 + b*(H psi).
//
// One thread owns one (site, rhs) pair, rhs fastest: thread tid = h*n + r.  The n threads of a site
// read the same link addresses (one L1 transaction, one HBM read per link per launch), the spinor
// loads of a warp are 128-bit and contiguous in memory for the centre site and for every neighbour
// direction inside a row of the site order.  Spin projection to half spinors happens in registers
// (table: DESIGN.md "Half-spinor projection"), so each direction costs 2 SU(3) x colour-vector
// products: 1320 flop per output site and RHS.
#include "wd_su3.cuh"

using namespace wdk;

namespace {

template <typename T>
struct HopArgs {
    const typename Vec<T>::type* in;   // half-lattice block of parity 1-par
    typename Vec<T>::type* out;        // half-lattice block of parity par
    const typename Vec<T>::type* in2;  // parity par, used by the XPAY epilogue
    const T* U;                        // native links of this precision and form
    const int32_t* nbr;                // [Vh][8] of parity par
    long Vh;
    int n;
    int par;
    T a, b;
};

// one direction: FWD: U_mu(x) psi(x+mu) with (1 - sg gamma);  !FWD: U_mu(x-mu)^dag psi(x-mu) with (1 + sg gamma)
template <typename T, int RECON, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void hop_dir(const HopArgs<T>& A, long h, int r, long nb, cx<T> (&acc)[12]) {
    constexpr int SIGMA = (FWD ? 1 : -1) * (DAG ? -1 : 1);
    const long stride = A.Vh * A.n;
    cx<T> psi[12], hs[6], chi[6], u[9];
    load_spinor(A.in, stride, nb * A.n + r, psi);
    if (FWD) load_link<RECON>(A.U + (long)(MU * 2 + A.par) * RECON * A.Vh, A.Vh, h, u);
    else     load_link<RECON>(A.U + (long)(MU * 2 + 1 - A.par) * RECON * A.Vh, A.Vh, nb, u);
    if (RECON == 12) rebuild_row3(u);
    project<MU, SIGMA>(psi, hs);
    su3_mul<!FWD>(u, hs, chi);
    accumulate<MU, SIGMA>(acc, chi);
}

template <typename T, int RECON, bool DAG, bool XPAY>
__global__ void __launch_bounds__(128) hop_kernel(const HopArgs<T> A) {
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= A.Vh * A.n) return;
    const long h = tid / A.n;
    const int r = (int)(tid - h * A.n);
    const long stride = A.Vh * A.n;
    const int4 n0 = __ldg(reinterpret_cast<const int4*>(A.nbr + h * WD_NDIR));
    const int4 n1 = __ldg(reinterpret_cast<const int4*>(A.nbr + h * WD_NDIR) + 1);
    cx<T> acc[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) { acc[k].re = 0; acc[k].im = 0; }
    if ((uint32_t)n0.x & WD_SITE_FROZEN) {  // SF: t = 0 stays zero
        store_spinor(A.out, stride, tid, acc);
        return;
    }
    hop_dir<T, RECON, 0, true, DAG>(A, h, r, n0.x, acc);
    hop_dir<T, RECON, 0, false, DAG>(A, h, r, n0.y, acc);
    hop_dir<T, RECON, 1, true, DAG>(A, h, r, n0.z, acc);
    hop_dir<T, RECON, 1, false, DAG>(A, h, r, n0.w, acc);
    hop_dir<T, RECON, 2, true, DAG>(A, h, r, n1.x, acc);
    hop_dir<T, RECON, 2, false, DAG>(A, h, r, n1.y, acc);
    hop_dir<T, RECON, 3, true, DAG>(A, h, r, n1.z, acc);
    hop_dir<T, RECON, 3, false, DAG>(A, h, r, n1.w, acc);
    if (XPAY) {
        cx<T> q[12];
        load_spinor(A.in2, stride, tid, q);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            acc[k].re = A.a * q[k].re + A.b * acc[k].re;
            acc[k].im = A.a * q[k].im + A.b * acc[k].im;
        }
    }
    store_spinor(A.out, stride, tid, acc);
}

template <typename T, int RECON>
void launch_t(wd_ctx* c, int dag, int n, int par, const void* in, void* out, const void* in2, double a, double b,
              const T* U) {
    HopArgs<T> A;
    A.in = (const typename Vec<T>::type*)in;
    A.out = (typename Vec<T>::type*)out;
    A.in2 = (const typename Vec<T>::type*)in2;
    A.U = U;
    A.nbr = c->d_nbr + (long)par * c->Vh * WD_NDIR;
    A.Vh = c->Vh;
    A.n = n;
    A.par = par;
    A.a = (T)a;
    A.b = (T)b;
    const long total = c->Vh * n;
    const int B = 128;
    const unsigned G = (unsigned)((total + B - 1) / B);
    const bool xpay = in2 != nullptr;
    if (dag) {
        if (xpay) hop_kernel<T, RECON, true, true><<<G, B, 0, c->stream>>>(A);
        else      hop_kernel<T, RECON, true, false><<<G, B, 0, c->stream>>>(A);
    } else {
        if (xpay) hop_kernel<T, RECON, false, true><<<G, B, 0, c->stream>>>(A);
        else      hop_kernel<T, RECON, false, false><<<G, B, 0, c->stream>>>(A);
    }
}

}  // namespace

int wd_hop_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const void* in, void* out,
                  const void* in2, double a, double b) {
    wd_prof_scope prof(c, prec == WD_F64 ? WD_PROF_HOP64 : WD_PROF_HOP32);
    if (prec == WD_F64) {
        if (recon == WD_LINK18) launch_t<double, 18>(c, dag, n, par, in, out, in2, a, b, c->d_U64[0]);
        else                    launch_t<double, 12>(c, dag, n, par, in, out, in2, a, b, c->d_U64[1]);
    } else {
        if (recon == WD_LINK18) launch_t<float, 18>(c, dag, n, par, in, out, in2, a, b, c->d_U32[0]);
        else                    launch_t<float, 12>(c, dag, n, par, in, out, in2, a, b, c->d_U32[1]);
    }
    WD_LAUNCH_CHECK(c);
    return WD_OK;
}
