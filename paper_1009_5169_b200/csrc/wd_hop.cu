// wd_hop.cu -- the multi-RHS even/odd Wilson hopping kernel (hot-path step a2; PAPER.md:80-84,
// "single-precision coefficient matrix D on the GPUs is also even/odd preconditioned").
//
//   (H psi)(x) = sum_mu (1 -+ gamma_mu) U_mu(x) psi(x+mu) + (1 +- gamma_mu) U_mu(x-mu)^dag psi(x-mu)
//   (upper sign D, lower sign D^dag) on ONE output parity, for all n_rhs columns in one launch,
//   optionally with a fused epilogue (out = a*in2 + b*(H psi), per-column inner products; see EPI_* below).
//
// This is the REGISTER kernel: operands go straight from global memory into registers.  It serves every site
// order and layout; where the layout is row-major and n_rhs >= 3 the staged kernel of wd_hop_tma.cu runs instead
// (WD_OPT_HOP_IMPL) and this one is the fallback and the reference for bit-equality.
//
// One thread owns one (site, rhs) pair, rhs fastest: thread tid = h*n + r.  The n threads of a site
// read the same link addresses (one L1 transaction, one HBM read per link per launch), the spinor
// loads of a warp are 128-bit and contiguous in memory for the centre site and for every neighbour
// direction inside a row of the site order.  Spin projection to half spinors happens in registers
// (table: DESIGN.md section 6a "Half-spinor projection"), so each direction costs 2 SU(3) x colour-vector
// products: 1320 flop per output site and RHS.
#include "wd_blas.cuh"
#include "wd_su3.cuh"

using namespace wdk;

namespace {

template <typename T>
struct HopArgs {
    const typename Vec<T>::type* in;   // half-lattice block of parity 1-par
    typename Vec<T>::type* out;        // half-lattice block of parity par
    const typename Vec<T>::type* in2;  // parity par, used by the xpay epilogue (EPI >= 1)
    const typename Vec<T>::type* in3;  // parity par, left operand of the fused <in3, out> (EPI == 2)
    wdblas::RedBuf rb;                 // per-column reduction scratch and scalar table (EPI >= 2)
    const double* done;                // nullable: the solver's "all columns converged" flag -> no-op launch
    const T* U;                        // native links of this precision and form
    const int32_t* nbr;                // [Vh][8] of parity par: PACKED site indices (block << lg) | offset
    uint32_t RB, lg;                   // native layout blocks of RB sites (wd_internal.h); 2^lg >= RB
    uint32_t Vh;
    uint32_t n;
    uint32_t par;
    uint32_t rev;                      // 1: CTA b works on block gridDim-1-b
    uint32_t total;                    // Vh * n  (wd_create bounds 12 * V/2 * max_rhs below 2^31: 32-bit indices)
    T a, b;
};

// one direction: FWD: U_mu(x) psi(x+mu) with (1 - sg gamma);  !FWD: U_mu(x-mu)^dag psi(x-mu) with (1 + sg gamma).
// (hb, ho) = layout block and offset of the output site, nb = packed index of the neighbour.
template <typename T, int RECON, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void hop_dir(const HopArgs<T>& A, uint32_t hb, uint32_t ho, uint32_t r, uint32_t nb,
                                        cx<T> (&acc)[12]) {
    constexpr int SIGMA = (FWD ? 1 : -1) * (DAG ? -1 : 1);
    constexpr uint32_t NCH = Vec<T>::NCH;
    const uint32_t nbb = nb >> A.lg, nbo = nb & ((1u << A.lg) - 1u);
    cx<T> psi[12], hs[6], chi[6], u[9];
    load_spinor(A.in + nbb * (NCH * A.RB * A.n), A.RB * A.n, nbo * A.n + r, psi);
    if (FWD) load_link<RECON>(A.U + (size_t)(MU * 2 + A.par) * RECON * A.Vh + (size_t)hb * RECON * A.RB, A.RB, ho, u);
    else     load_link<RECON>(A.U + (size_t)(MU * 2 + 1 - A.par) * RECON * A.Vh + (size_t)nbb * RECON * A.RB, A.RB, nbo, u);
    if (RECON == 12) rebuild_row3(u);
    project<MU, SIGMA>(psi, hs);
    su3_mul<!FWD>(u, hs, chi);
    accumulate<MU, SIGMA>(acc, chi);
}

// Epilogues fused into the hop (one kernel boundary per global reduction):
//   EPI_NONE  out = H in
//   EPI_XPAY  out = a in2 + b H in
//   EPI_SIGMA EPI_XPAY, then sigma_i = <in3_i, out_i> per column  -> alpha_i = rho_i / sigma_i   (in3 = r~, out = v)
//   EPI_OMEGA EPI_XPAY, then <out_i, in2_i>, <out_i, out_i>       -> omega_i                     (in2 = s,  out = t)
// Each CTA leaves one partial per column and value; a tiny finalize_partials_kernel (one block per item)
// adds them in a fixed order and runs the scalar recurrence, so no dot-product kernel re-reads the vectors.
enum { EPI_NONE = 0, EPI_XPAY = 1, EPI_SIGMA = 2, EPI_OMEGA = 3 };

// Launch shape: S sites x n columns per CTA (column fastest), S = WD_OPT_HOP*_SITES.
template <typename T, int RECON, bool DAG, int EPI, int MAXREG>
__global__ void __maxnreg__(MAXREG) hop_kernel(const HopArgs<T> A) {
    if (A.done != nullptr && *A.done != 0.0) return;
    const uint32_t tid = (A.rev ? gridDim.x - 1 - blockIdx.x : blockIdx.x) * blockDim.x + threadIdx.x;
    const bool in_range = tid < A.total;
    if (EPI < EPI_SIGMA && !in_range) return;
    const uint32_t h = in_range ? tid / A.n : 0u;
    const uint32_t r = tid - (tid / A.n) * A.n;
    const uint32_t hb = h / A.RB, ho = h - hb * A.RB;        // layout block and offset of this site
    const uint32_t rbn = A.RB * A.n;                          // chunk stride inside a layout block
    const uint32_t own = hb * (Vec<T>::NCH * rbn);            // first element of the block
    const uint32_t eo = ho * A.n + r;                         // this (site, column) inside a chunk
    const int4 n0 = __ldg(reinterpret_cast<const int4*>(A.nbr) + 2 * h);
    const int4 n1 = __ldg(reinterpret_cast<const int4*>(A.nbr) + 2 * h + 1);
    cx<T> acc[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) { acc[k].re = 0; acc[k].im = 0; }
    const bool frozen = ((uint32_t)n0.x & WD_SITE_FROZEN) != 0;  // SF: t = 0 stays zero
    if (EPI < EPI_SIGMA && frozen) {
        store_spinor(A.out + own, rbn, eo, acc);
        return;
    }
    // per-thread partial sums over the 12 components of ONE site and column in working precision
    // (fp32: 24-72 products); everything across threads is added in fp64 (wd_blas.cuh)
    [[maybe_unused]] T sums[3] = {0, 0, 0};
    if (in_range && !frozen) {
        if (EPI >= EPI_XPAY) {  // the epilogue's operands: ask L2 for them now, they are read after the eight directions
#pragma unroll
            for (uint32_t c = 0; c < Vec<T>::NCH; ++c) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in2 + own + c * rbn + eo));
                if (EPI == EPI_SIGMA) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in3 + own + c * rbn + eo));
            }
        }
        if constexpr (sizeof(T) == 4) {
            // fp32: the order in which the z-march kernel (wd_hop_zm.cu) consumes its units, so that the two
            // kernels agree bit for bit
            hop_dir<T, RECON, 3, true, DAG>(A, hb, ho, r, n1.z, acc);
            hop_dir<T, RECON, 3, false, DAG>(A, hb, ho, r, n1.w, acc);
            hop_dir<T, RECON, 2, false, DAG>(A, hb, ho, r, n1.y, acc);
            hop_dir<T, RECON, 1, false, DAG>(A, hb, ho, r, n0.w, acc);
            hop_dir<T, RECON, 1, true, DAG>(A, hb, ho, r, n0.z, acc);
            hop_dir<T, RECON, 0, false, DAG>(A, hb, ho, r, n0.y, acc);
            hop_dir<T, RECON, 0, true, DAG>(A, hb, ho, r, n0.x, acc);
            hop_dir<T, RECON, 2, true, DAG>(A, hb, ho, r, n1.x, acc);
        } else {
            // fp64: the order of wd_hop_tma.cu's units (the staged kernel that serves fp64)
            hop_dir<T, RECON, 0, true, DAG>(A, hb, ho, r, n0.x, acc);
            hop_dir<T, RECON, 0, false, DAG>(A, hb, ho, r, n0.y, acc);
            hop_dir<T, RECON, 1, true, DAG>(A, hb, ho, r, n0.z, acc);
            hop_dir<T, RECON, 1, false, DAG>(A, hb, ho, r, n0.w, acc);
            hop_dir<T, RECON, 2, true, DAG>(A, hb, ho, r, n1.x, acc);
            hop_dir<T, RECON, 2, false, DAG>(A, hb, ho, r, n1.y, acc);
            hop_dir<T, RECON, 3, true, DAG>(A, hb, ho, r, n1.z, acc);
            hop_dir<T, RECON, 3, false, DAG>(A, hb, ho, r, n1.w, acc);
        }
        if (EPI >= EPI_XPAY) {
            cx<T> q[12];
            load_spinor(A.in2 + own, rbn, eo, q);
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                acc[k].re = fma(A.b, acc[k].re, A.a * q[k].re);
                acc[k].im = fma(A.b, acc[k].im, A.a * q[k].im);
            }
            if (EPI == EPI_OMEGA) {  // <t, s>, <t, t> with t = acc, s = q
#pragma unroll
                for (int k = 0; k < 12; ++k) {
                    sums[0] = fma(acc[k].re, q[k].re, sums[0]);  sums[0] = fma(acc[k].im, q[k].im, sums[0]);
                    sums[1] = fma(acc[k].re, q[k].im, sums[1]);  sums[1] = fma(-acc[k].im, q[k].re, sums[1]);
                    sums[2] = fma(acc[k].re, acc[k].re, sums[2]); sums[2] = fma(acc[k].im, acc[k].im, sums[2]);
                }
            }
        }
        if (EPI == EPI_SIGMA) {  // <r~, v> with v = acc
            cx<T> q[12];
            load_spinor(A.in3 + own, rbn, eo, q);
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                sums[0] = fma(q[k].re, acc[k].re, sums[0]);  sums[0] = fma(q[k].im, acc[k].im, sums[0]);
                sums[1] = fma(q[k].re, acc[k].im, sums[1]);  sums[1] = fma(-q[k].im, acc[k].re, sums[1]);
            }
        }
    }
    if (in_range) store_spinor(A.out + own, rbn, eo, acc);
    if (EPI == EPI_SIGMA) {  // block partials; finalize_partials_kernel follows on the stream
        double s2[2] = {(double)sums[0], (double)sums[1]};
        wdblas::block_partials<2>(s2, (int)A.n, A.rb);
    } else if (EPI == EPI_OMEGA) {
        double s3[3] = {(double)sums[0], (double)sums[1], (double)sums[2]};
        wdblas::block_partials<3>(s3, (int)A.n, A.rb);
    }
}

template <typename T, int RECON, int MAXREG>
void launch_r(wd_ctx* c, const HopArgs<T>& A, int dag, int epi, unsigned G, unsigned B) {
#define WD_HOP_CASE(D, E) hop_kernel<T, RECON, D, E, MAXREG><<<G, B, 0, c->stream>>>(A)
    if (dag) {
        if (epi == EPI_NONE) WD_HOP_CASE(true, EPI_NONE);
        else if (epi == EPI_XPAY) WD_HOP_CASE(true, EPI_XPAY);
        else if constexpr (sizeof(T) == 4) { if (epi == EPI_SIGMA) WD_HOP_CASE(true, EPI_SIGMA); else WD_HOP_CASE(true, EPI_OMEGA); }
    } else {
        if (epi == EPI_NONE) WD_HOP_CASE(false, EPI_NONE);
        else if (epi == EPI_XPAY) WD_HOP_CASE(false, EPI_XPAY);
        else if constexpr (sizeof(T) == 4) { if (epi == EPI_SIGMA) WD_HOP_CASE(false, EPI_SIGMA); else WD_HOP_CASE(false, EPI_OMEGA); }
    }
#undef WD_HOP_CASE
}

template <typename T, int RECON>
int launch_t(wd_ctx* c, int dag, int n, int par, const wd_hop_ops& o, const T* U) {
    HopArgs<T> A;
    A.in = (const typename Vec<T>::type*)o.in;
    A.out = (typename Vec<T>::type*)o.out;
    A.in2 = (const typename Vec<T>::type*)o.in2;
    A.in3 = (const typename Vec<T>::type*)o.in3;
    A.rb = wdblas::RedBuf{c->d_scal, c->d_partials, c->d_ticket};
    A.done = o.check_done ? c->d_scal + wdblas::G_DONE : nullptr;
    A.U = U;
    A.nbr = c->d_nbr + (long)par * c->Vh * WD_NDIR;
    A.Vh = (uint32_t)c->Vh;
    A.RB = c->RB;
    A.lg = c->rb_lg;
    A.n = (uint32_t)n;
    A.par = (uint32_t)par;
    A.rev = o.rev ? 1u : 0u;
    A.total = (uint32_t)(c->Vh * n);
    A.a = (T)o.a;
    A.b = (T)o.b;
    const bool f64 = sizeof(T) == 8;
    // CTA = `sites` sites x n columns.  Measured at 24^4 (fp32, R=12): about 64-160 threads per CTA is best for
    // every n_rhs (n=5: 32 sites, n=8: 8-16, n=12, 16: 8), and 64 registers (more CTAs per SM) from n = 3 up.
    int sites = c->opt[f64 ? WD_OPT_HOP64_SITES : WD_OPT_HOP32_SITES];
    const bool fused = o.epi >= EPI_SIGMA;
    if (sites == 0) {
        sites = 32;
        if (!f64)
            for (int s = 8; s < 32; s <<= 1)
                if ((s * n) % 32 == 0 && s * n >= 64) { sites = s; break; }
        if (f64) sites = 16;
    }
    // fused reductions: exactly 32 sites per CTA.  B = 32 n is a multiple of 32 (the block reduction shuffles whole
    // warps) and at most 512, and the grid is ceil(V/2 / 32) blocks, which is what the partial-sum buffer is sized
    // for (wd_ctx.cu partial_doubles: n * K * G doubles are written); the option does not apply to these launches.
    if (fused) sites = 32;
    while (sites * n > (fused ? 512 : 1024) && sites > 1) sites >>= 1;
    // the smallest compiled variant needs 128 (fp64) / 64 (fp32) registers per thread: keep one CTA within an SM
    while ((long)sites * n * (f64 ? 128 : 64) > 65536 && sites > 1) sites >>= 1;
    const unsigned B = (unsigned)(sites * n);
    const unsigned G = (A.total + B - 1) / B;
    if (fused && (size_t)G * 3 * WD_MAX_RHS > c->partial_doubles) return wd_fail(c, WD_EINVAL, "hop: reduction scratch too small for this grid");
    // largest compiled register budget that the option allows and that lets one CTA of B threads fit
    int regs = c->opt[f64 ? WD_OPT_HOP64_REGS : WD_OPT_HOP32_REGS];
    if (regs == 0) regs = f64 ? 168 : ((n <= 2 || RECON == 18) ? 128 : 64);  // 18-real links: 64 registers spill
    if ((long)regs * B > 65536) regs = (int)(65536 / B);
    if constexpr (sizeof(T) == 8) {
        if (regs >= 168) launch_r<T, RECON, 168>(c, A, dag, o.epi, G, B);
        else             launch_r<T, RECON, 128>(c, A, dag, o.epi, G, B);
    } else {
        if (regs >= 128) launch_r<T, RECON, 128>(c, A, dag, o.epi, G, B);
        else             launch_r<T, RECON, 64>(c, A, dag, o.epi, G, B);
    }
    if (o.epi == EPI_SIGMA)
        wdblas::finalize_partials_kernel<2, wdblas::K_SIGMA><<<2 * n, 256, 0, c->stream>>>(n, G, A.rb, c->d_totals);
    else if (o.epi == EPI_OMEGA)
        wdblas::finalize_partials_kernel<3, wdblas::K_OMEGA><<<3 * n, 256, 0, c->stream>>>(n, G, A.rb, c->d_totals);
    if (o.epi >= EPI_SIGMA) c->launches++;
    return WD_OK;
}

}  // namespace

int wd_hop_launch_ex(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o) {
    wd_prof_scope prof(c, prec == WD_F64 ? WD_PROF_HOP64 : WD_PROF_HOP32);
    if (o.epi >= EPI_SIGMA && prec != WD_F32) return wd_fail(c, WD_EINVAL, "fused reductions are fp32 only");
    // staged kernel where it applies (row-major layout) and pays: with 1-2 columns a group of rows gives it too few
    // consumer threads (24^4 fp32: 41 us against 33 us at n = 2; 71 against 76 at n = 5; 146 against 151 at n = 12)
    if (o.epi == 4) {   // xpay + <t,s>, <t,t>, <rt,s>, <rt,t> (merged-update schedule): plain fp32 operands, z-march kernel only
        const int rc = (prec == WD_F32 && o.storage == 0 && n >= 3) ? wd_hop_zm_launch(c, prec, recon, dag, n, par, o) : 1;
        if (rc > 0) return wd_fail(c, WD_EINVAL, "hop: the seven-sum epilogue needs the z-march kernel");
        if (rc == WD_OK) WD_LAUNCH_CHECK(c);
        return rc;
    }
    if (prec == WD_F32P || o.storage == 2) {   // P32 (two sites per thread): served by the z-march kernel only
        wd_hop_ops o2 = o;
        o2.storage = 2;
        const int rc = wd_hop_zm_launch(c, WD_F32, recon, dag, n, par, o2);
        if (rc > 0) return wd_fail(c, WD_EINVAL, "hop: WD_F32P needs the z-march kernel (row-major layout, a shape that fits shared memory)");
        if (rc == WD_OK) WD_LAUNCH_CHECK(c);
        return rc;
    }
    if (o.storage == 1) {   // 16-bit storage: served by the z-march kernel only
        const int rc = n >= 3 ? wd_hop_zm_launch(c, prec, recon, dag, n, par, o) : 1;
        if (rc > 0) return wd_fail(c, WD_EINVAL, "hop: the 16-bit storage format needs the z-march kernel (row-major layout, n_rhs >= 3)");
        if (rc == WD_OK) WD_LAUNCH_CHECK(c);
        return rc;
    }
    if (c->opt[WD_OPT_HOP_IMPL] >= 1 && n >= 3) {
        int rc = 1;
        const int impl = c->opt[WD_OPT_HOP_IMPL];
        if (impl == 3 || (impl == 2 && (prec != WD_F32 || wd_hop_zm_preferred(c, recon, n)))) rc = wd_hop_zm_launch(c, prec, recon, dag, n, par, o);
        if (rc > 0) rc = wd_hop_tma_launch(c, prec, recon, dag, n, par, o);
        if (rc <= 0) {
            if (rc == WD_OK) WD_LAUNCH_CHECK(c);
            return rc;
        }
    }
    int rc;
    if (prec == WD_F64) {
        if (recon == WD_LINK18) rc = launch_t<double, 18>(c, dag, n, par, o, c->d_U64[0]);
        else                    rc = launch_t<double, 12>(c, dag, n, par, o, c->d_U64[1]);
    } else {
        if (recon == WD_LINK18) rc = launch_t<float, 18>(c, dag, n, par, o, c->d_U32[0]);
        else                    rc = launch_t<float, 12>(c, dag, n, par, o, c->d_U32[1]);
    }
    if (rc) return rc;
    WD_LAUNCH_CHECK(c);
    return WD_OK;
}

// The kernel the dispatch above picks for plain operands (storage 0, epilogues 0-3): keep the two in step.
int wd_hop_kernel_for(const wd_ctx* c, int prec, int recon, int n) {
    const int impl = c->opt[WD_OPT_HOP_IMPL];
    if (impl >= 1 && n >= 3) {
        if ((impl == 3 || (impl == 2 && (prec != WD_F32 || wd_hop_zm_preferred(c, recon, n)))) && prec == WD_F32 &&
            wd_hop_zm_serves(c, recon, n, 0))
            return WD_HOP_KERNEL_ZMARCH;
        if (wd_hop_tma_serves(c, prec, recon, n)) return WD_HOP_KERNEL_RING;
    }
    return WD_HOP_KERNEL_REGISTER;
}

int wd_hop_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const void* in, void* out,
                  const void* in2, double a, double b) {
    wd_hop_ops o;
    o.in = in; o.out = out; o.in2 = in2; o.in3 = nullptr;
    o.a = a; o.b = b;
    o.epi = in2 ? EPI_XPAY : EPI_NONE;
    o.check_done = false;
    o.rev = 0;
    o.storage = 0;
    return wd_hop_launch_ex(c, prec, recon, dag, n, par, o);
}
