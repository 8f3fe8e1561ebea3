// wd_hop_tma.cu -- the multi-RHS Wilson hopping kernel with its operands staged through shared memory by
// the bulk-copy engine (TMA, cp.async.bulk + mbarrier) -- hot-path step a2, the B200 form of wd_hop.cu.
//
// Why it exists: the register kernel (wd_hop.cu) loads one direction at a time into registers; with 4-7 warps
// per scheduler nothing covers the load latency, so memory time and arithmetic time largely ADD (ncu: long-
// scoreboard stalls 7 per issue, issue slots 41 % busy; ablations in DESIGN.md section 6).  Here one persistent CTA
// per SM runs a producer warp that streams whole lattice rows into a ring of shared-memory slots with
// cp.async.bulk (no registers, no LSU instructions, ~150 KB in flight per SM), and consumer warps (one thread
// per site and column) that only ever wait on an mbarrier, read shared memory and do arithmetic.
//
// It needs the row-major native layout (wd_layout.cu, RB = Lx/2): there a lattice row is contiguous with all its
// chunks, so every piece a unit needs is ONE bulk copy of whole rows (about 15 copies per group).  In the earlier
// chunk-major layout a group took about 60 copies of 1-4 KB, and at a measured ~85 ns of issue cost per copy the
// producer alone needed 49 us per launch, longer than the consumers' arithmetic.
//
// Measured (B200, 24^4, n_rhs = 5, fp32, L2-cold, standalone): 71 us (12-real links) / 70 us (18-real), results bit
// for bit those of the register kernel, which takes 70 us in the chunk-major layout and 76 us in this one.  Inside
// the solver (half of the launches carry the fused xpay / inner-product epilogues) this kernel averages 84 us per
// launch against 91 us for the register kernel.  Where the time goes: producers alone 43 us,
// consumers alone 51 us (32 us of pure issue time), together 70: the ring is one group deep (it takes the whole
// 227 KB of shared memory, one CTA per SM), so the fourth small unit of a group and the next XY unit arrive late
// (mbarrier waits: 18 % of the stall samples).
//
// A note for whoever touches the producers: keep their code small.  An earlier version with fully unrolled copy
// loops (fp64, 12 chunks) made ptxas run out of uniform registers and emit R2UR.FILL spills around the UBLKCP
// instructions; that build raised "illegal memory access" on every fp64 launch although every address and size
// checked out (cuobjdump -sass | grep R2UR.FILL should stay empty).
//
// Geometry (linear site order only): a half-lattice index is h = xh + Lxh*(y + Ly*(z + Lz*t)), xh = x/2.
// A "row" is the Lxh sites of fixed (y,z,t); neighbours in +-y, +-z, +-t of a row are the row with the
// same xh at the shifted (y,z,t); neighbours in +-x are in the row with the same (y,z,t) of the other
// parity at xh or xh+-1 (which one depends on the parity of y+z+t+par).  So no neighbour table is read.
// Work item = a group of RG consecutive rows in y (S = RG*Lxh sites, S*n consumer threads).  Per group the
// producers issue 5 units:  XY (input rows y0-1 .. y0+RG, links x+ x- y+ y-), Z+, Z-, T+, T- (RG input rows
// and one link array each).  Ring: one big slot for XY units and three small slots for the others.
#include "wd_blas.cuh"
#include "wd_su3.cuh"
#include "wd_tma.cuh"

using namespace wdk;
using namespace wdtma;

namespace {

enum { EPI_NONE = 0, EPI_XPAY = 1, EPI_SIGMA = 2, EPI_OMEGA = 3 };

// ---- arguments -------------------------------------------------------------------------------------
template <typename T>
struct TmaArgs {
    const typename Vec<T>::type* in;   // half-lattice block of parity 1-par
    typename Vec<T>::type* out;        // half-lattice block of parity par
    const typename Vec<T>::type* in2;  // xpay operand (EPI >= 1)
    const typename Vec<T>::type* in3;  // left operand of <in3, out> (EPI == 2)
    const T* U;                        // native links of this precision and form
    wdblas::RedBuf rb;
    const double* done;
    uint32_t Lxh, Ly, Lz, Lt;
    uint32_t Vh, n, par, total;        // total = Vh * n
    uint32_t RG, S;                    // rows per group, sites per group = RG * Lxh
    uint32_t groups;                   // (Ly / RG) * Lz * Lt
    uint32_t g_first;                  // groups [0, g_first) are the frozen t = 0 slice (Schroedinger functional), else 0
    uint32_t big_vecs, small_vecs;     // slot sizes in 16-byte units
    uint32_t NS;                       // number of small slots in the ring (3..7)
    uint32_t NP;                       // producer warps: 2 when they fit beside the consumers, else 1
    T a, b;
};

__device__ __forceinline__ uint32_t wrap_inc(uint32_t v, uint32_t L) { return v + 1 == L ? 0u : v + 1; }
__device__ __forceinline__ uint32_t wrap_dec(uint32_t v, uint32_t L) { return v == 0 ? L - 1 : v - 1; }

// ---- producer side ------------------------------------------------------------------------------------
// In the row-major native layout (wd_layout.cu with RB = Lx/2) a lattice row is contiguous with all its chunks:
// NCH * rowB bytes of spinor, lrowB = Lxh * R * sizeof(T) bytes of link per (mu, parity).  So every piece a unit
// needs is ONE bulk copy of whole rows: 5-8 copies for the XY unit, 2 for the others (about 15 per group; in the
// chunk-major layout it took about 60, and at ~85 ns of issue cost per copy the producer was the bottleneck).
// The producer warp builds the copy list lane-parallel: lane k owns copy k.
struct CopyDesc {
    char* dst;
    const char* src;
    uint32_t bytes;  // 0 = nothing to copy
};

template <typename T, int RECON>
__device__ void produce_xy(const TmaArgs<T>& A, uint32_t lane, uint32_t y0, uint32_t z, uint32_t t, uint32_t q, char* ring,
                              uint64_t* full, uint64_t* empty) {
    constexpr uint32_t NCH = Vec<T>::NCH;
    const uint32_t rowB = A.Lxh * A.n * 16 * NCH;                   // bytes of one spinor row (all chunks)
    const uint32_t lrowB = A.Lxh * RECON * (uint32_t)sizeof(T);     // bytes of one row of one link array
    const uint32_t RG = A.RG;
    const uint32_t zt = z + A.Lz * t;
    const uint32_t row0 = y0 + A.Ly * zt;
    const char* in = reinterpret_cast<const char*>(A.in);
    const char* U = reinterpret_cast<const char*>(A.U);
    const size_t ublk = (size_t)RECON * A.Vh * sizeof(T);           // bytes of one (mu, parity) link array
    // ---- XY unit -> big slot (use q): rows y0-1 .. y0+RG, links x+ x- y+ y-
    {
        mbar_wait(&empty[0], (q & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&full[0], (RG + 2) * rowB + 4 * RG * lrowB);
        __syncwarp();
        char* B = ring;
        char* L = B + (size_t)(RG + 2) * rowB;
        const bool lo = y0 == 0, hi = y0 + RG == A.Ly;   // the halo row below / above wraps around in y
        const uint32_t rm = (lo ? A.Ly - 1 : y0 - 1) + A.Ly * zt;
        const uint32_t rp = (hi ? 0 : y0 + RG) + A.Ly * zt;
        CopyDesc d;
        d.bytes = 0;
        if (lane == 0) {         // rows y0 .. y0+RG-1 with whichever halo rows are contiguous with them
            const uint32_t first = lo ? 1u : 0u, nrows = RG + (lo ? 0u : 1u) + (hi ? 0u : 1u);
            d.dst = B + (size_t)first * rowB; d.src = in + (size_t)(row0 - (lo ? 0u : 1u)) * rowB; d.bytes = nrows * rowB;
        } else if (lane == 1) {  // halo row below, when it wraps
            d.dst = B; d.src = in + (size_t)rm * rowB; d.bytes = lo ? rowB : 0u;
        } else if (lane == 2) {  // halo row above, when it wraps
            d.dst = B + (size_t)(RG + 1) * rowB; d.src = in + (size_t)rp * rowB; d.bytes = hi ? rowB : 0u;
        } else if (lane == 3) {  // x+: U_x(x) on the output rows
            d.dst = L; d.src = U + (size_t)(0 + A.par) * ublk + (size_t)row0 * lrowB; d.bytes = RG * lrowB;
        } else if (lane == 4) {  // x-: U_x(x - x^) lives on the same rows of the other parity
            d.dst = L + (size_t)RG * lrowB; d.src = U + (size_t)(0 + 1 - A.par) * ublk + (size_t)row0 * lrowB; d.bytes = RG * lrowB;
        } else if (lane == 5) {  // y+: U_y(x)
            d.dst = L + (size_t)2 * RG * lrowB; d.src = U + (size_t)(2 + A.par) * ublk + (size_t)row0 * lrowB; d.bytes = RG * lrowB;
        } else if (lane == 6) {  // y-: U_y(x - y^) on rows y0-1 .. y0+RG-2 of the other parity (one piece unless row y0-1 wraps)
            d.dst = L + (size_t)3 * RG * lrowB + (lo ? lrowB : 0u);
            d.src = U + (size_t)(2 + 1 - A.par) * ublk + (size_t)(lo ? row0 : row0 - 1) * lrowB;
            d.bytes = (lo ? RG - 1 : RG) * lrowB;
        } else if (lane == 7) {
            d.dst = L + (size_t)3 * RG * lrowB; d.src = U + (size_t)(2 + 1 - A.par) * ublk + (size_t)rm * lrowB; d.bytes = lo ? lrowB : 0u;
        }
        if (d.bytes) bulk_g2s(d.dst, d.src, d.bytes, &full[0]);
    }
}

template <typename T, int RECON>
__device__ void produce_small(const TmaArgs<T>& A, uint32_t lane, uint32_t y0, uint32_t z, uint32_t t, uint32_t q, char* ring,
                              uint64_t* full, uint64_t* empty) {
    constexpr uint32_t NCH = Vec<T>::NCH;
    const uint32_t rowB = A.Lxh * A.n * 16 * NCH;                   // bytes of one spinor row (all chunks)
    const uint32_t lrowB = A.Lxh * RECON * (uint32_t)sizeof(T);     // bytes of one row of one link array
    const uint32_t RG = A.RG;
    const uint32_t zt = z + A.Lz * t;
    const uint32_t row0 = y0 + A.Ly * zt;
    const char* in = reinterpret_cast<const char*>(A.in);
    const char* U = reinterpret_cast<const char*>(A.U);
    const size_t ublk = (size_t)RECON * A.Vh * sizeof(T);           // bytes of one (mu, parity) link array
    // ---- Z+, Z-, T+, T- units -> small slots: RG rows of the shifted plane and one link array
    const size_t bigB = (size_t)A.big_vecs * 16, smallB = (size_t)A.small_vecs * 16;
#pragma unroll 1
    for (uint32_t u = 0; u < 4; ++u) {
        const uint32_t m = 4 * q + u, slot = 1 + m % A.NS, use = m / A.NS;
        mbar_wait(&empty[slot], (use & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&full[slot], RG * rowB + RG * lrowB);
        __syncwarp();
        char* B = ring + bigB + (size_t)(slot - 1) * smallB;
        uint32_t zz = z, tt = t;
        if (u == 0) zz = wrap_inc(z, A.Lz);
        else if (u == 1) zz = wrap_dec(z, A.Lz);
        else if (u == 2) tt = wrap_inc(t, A.Lt);
        else tt = wrap_dec(t, A.Lt);
        const uint32_t rn = y0 + A.Ly * (zz + A.Lz * tt);
        const bool fwd = (u & 1) == 0;
        if (lane == 0) bulk_g2s(B, in + (size_t)rn * rowB, RG * rowB, &full[slot]);
        else if (lane == 1)
            bulk_g2s(B + (size_t)RG * rowB,
                     U + (size_t)((2 + (u >> 1)) * 2 + (fwd ? A.par : 1 - A.par)) * ublk + (size_t)(fwd ? row0 : rn) * lrowB,
                     RG * lrowB, &full[slot]);
    }
}

// ---- consumer side ------------------------------------------------------------------------------------
__device__ __forceinline__ void lds_spinor(const float4* __restrict__ sp, uint32_t stride, uint32_t e, cx<float> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float4 v = sp[c * stride + e];
        psi[2 * c].re = v.x; psi[2 * c].im = v.y; psi[2 * c + 1].re = v.z; psi[2 * c + 1].im = v.w;
    }
}
__device__ __forceinline__ void lds_spinor(const double2* __restrict__ sp, uint32_t stride, uint32_t e, cx<double> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        const double2 v = sp[c * stride + e];
        psi[c].re = v.x; psi[c].im = v.y;
    }
}
// staged link array `L` (S sites per chunk), site index `site`
template <int RECON>
__device__ __forceinline__ void lds_link(const float4* __restrict__ L, uint32_t S, uint32_t site, cx<float> (&u)[9]) {
#pragma unroll
    for (int c = 0; c < (RECON == 18 ? 4 : 3); ++c) {
        const float4 v = L[c * S + site];
        u[2 * c].re = v.x; u[2 * c].im = v.y; u[2 * c + 1].re = v.z; u[2 * c + 1].im = v.w;
    }
    if (RECON == 18) {
        const float2 w = reinterpret_cast<const float2*>(L + 4 * S)[site];
        u[8].re = w.x; u[8].im = w.y;
    }
}
template <int RECON>
__device__ __forceinline__ void lds_link(const double2* __restrict__ L, uint32_t S, uint32_t site, cx<double> (&u)[9]) {
#pragma unroll
    for (int c = 0; c < (RECON == 18 ? 9 : 6); ++c) {
        const double2 v = L[c * S + site];
        u[c].re = v.x; u[c].im = v.y;
    }
}

// one direction from staged operands: spinor at (sp, stride, e), link array L at `site`
template <typename T, int RECON, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void dir_smem(const typename Vec<T>::type* sp, uint32_t stride, uint32_t e,
                                         const typename Vec<T>::type* L, uint32_t S, uint32_t site, cx<T> (&acc)[12]) {
    constexpr int SIGMA = (FWD ? 1 : -1) * (DAG ? -1 : 1);
    cx<T> psi[12], hs[6], chi[6], u[9];
    lds_spinor(sp, stride, e, psi);
    lds_link<RECON>(L, S, site, u);
    if (RECON == 12) rebuild_row3(u);
    project<MU, SIGMA>(psi, hs);
    su3_mul<!FWD>(u, hs, chi);
    accumulate<MU, SIGMA>(acc, chi);
}

// ---- the kernel -----------------------------------------------------------------------------------------
// grid = min(groups, SMs) persistent CTAs; block = consumer warps (S*n threads, rounded up) + 1 or 2 producer warps
// (at n = 5: 15 + 1 = 16 warps, so the consumers get 128 registers; a second producer warp bought nothing there).
// dynamic smem: 128 bytes of mbarriers, then the ring: [big slot][NS small slots], NS = as many as fit (>= 3).
template <typename T, int RECON, bool DAG, int EPI, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) hop_tma_kernel(const TmaArgs<T> A) {
    typedef typename Vec<T>::type vec;
    if (A.done != nullptr && *A.done != 0.0) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* empty = full + 8;   // up to 1 + 7 slots
    char* ring = reinterpret_cast<char*>(smem) + 128;
    const uint32_t nct = A.S * A.n;            // consumer threads
    const uint32_t ncw = (nct + 31) >> 5;      // consumer warps
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < 1 + A.NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], ncw); }
        mbar_fence_init();
    }
    __syncthreads();
    const uint32_t gy = A.Ly / A.RG;
    [[maybe_unused]] double dsum[3] = {0.0, 0.0, 0.0};

    if (warp >= ncw) {
        // ================= producer warp: every bulk copy of this CTA's groups ======================
        uint32_t q = 0;
        for (uint32_t g = A.g_first + blockIdx.x; g < A.groups; g += gridDim.x) {
            const uint32_t yg = g % gy, zt = g / gy, z = zt % A.Lz, t = zt / A.Lz;
            // one producer warp issues both slot classes; with two, warp ncw takes the XY units and warp ncw+1 the others
            if (A.NP == 1 || warp == ncw) produce_xy<T, RECON>(A, lane, yg * A.RG, z, t, q, ring, full, empty);
            if (A.NP == 1 || warp != ncw) produce_small<T, RECON>(A, lane, yg * A.RG, z, t, q, ring, full, empty);
            ++q;
        }
    } else {
        // ================= consumers: thread i = (site s of the group, column r) =========================
        const uint32_t i = threadIdx.x;
        const bool active = i < nct;
        const uint32_t s = i / A.n, r = i - s * A.n;
        const uint32_t j = s / A.Lxh, xh = s - j * A.Lxh;   // row inside the group, site inside the row
        constexpr uint32_t NCH = Vec<T>::NCH;
        const uint32_t rowV = A.Lxh * A.n, RG = A.RG;
        const uint32_t lrowV = A.Lxh * RECON * (uint32_t)sizeof(T) / 16;   // 16-byte units of one link row
        const vec* bigS = reinterpret_cast<const vec*>(ring);
        const vec* bigL = bigS + (size_t)(RG + 2) * NCH * rowV;
        const uint32_t e0 = xh * A.n + r;                    // this (site, column) inside a chunk of a row
        uint32_t q = 0;
        if (active) {  // SF: the stored t = 0 slice stays zero
            cx<T> zero[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) { zero[k].re = 0; zero[k].im = 0; }
            for (uint32_t g = blockIdx.x; g < A.g_first; g += gridDim.x) {
                const uint32_t row = (g % gy) * RG + A.Ly * (g / gy) + j;
                store_spinor(A.out + (size_t)row * NCH * rowV, rowV, e0, zero);
            }
        }
        for (uint32_t g = A.g_first + blockIdx.x; g < A.groups; g += gridDim.x) {
            const uint32_t yg = g % gy, zt = g / gy, z = zt % A.Lz, t = zt / A.Lz;
            const uint32_t y0 = yg * RG;
            const size_t own = (size_t)(y0 + A.Ly * zt + j) * NCH * rowV;   // first element of this site's row
            cx<T> acc[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) { acc[k].re = 0; acc[k].im = 0; }
            // the epilogue's operands are only needed after all eight directions: ask L2 for them now, so that the
            // loads at the end of the group do not wait on DRAM (they cannot be hoisted: no registers to hold them)
            if (EPI >= EPI_XPAY && active) {
#pragma unroll
                for (uint32_t c = 0; c < NCH; ++c) {
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in2 + own + c * rowV + e0));
                    if (EPI == EPI_SIGMA) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in3 + own + c * rowV + e0));
                }
            }
            // ---- XY unit
            mbar_wait(&full[0], q & 1);
            if (active) {
                const uint32_t b = (y0 + j + z + t + A.par) & 1;
                const uint32_t xp = b ? wrap_inc(xh, A.Lxh) : xh;   // xh of the +x neighbour
                const uint32_t xm = b ? xh : wrap_dec(xh, A.Lxh);   // xh of the -x neighbour
                const vec* rowc = bigS + (size_t)(j + 1) * NCH * rowV;     // staged rows: 0 = y0-1, 1.. = y0.., RG+1 = y0+RG
                const vec* lk = bigL + (size_t)j * lrowV;                  // link arrays: x+ | x- | y+ | y-, RG rows each
                dir_smem<T, RECON, 0, true, DAG>(rowc, rowV, xp * A.n + r, lk, A.Lxh, xh, acc);
                dir_smem<T, RECON, 0, false, DAG>(rowc, rowV, xm * A.n + r, lk + (size_t)RG * lrowV, A.Lxh, xm, acc);
                dir_smem<T, RECON, 1, true, DAG>(rowc + NCH * rowV, rowV, e0, lk + (size_t)2 * RG * lrowV, A.Lxh, xh, acc);
                dir_smem<T, RECON, 1, false, DAG>(rowc - NCH * rowV, rowV, e0, lk + (size_t)3 * RG * lrowV, A.Lxh, xh, acc);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[0]);
            // ---- Z+, Z-, T+, T- units
            [[maybe_unused]] cx<T> qv[12];   // the xpay operand: requested before the wait for the last unit
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t m = 4 * q + u, slot = 1 + m % A.NS, use = m / A.NS;
                // (fp32 only: in fp64 the 24 extra doubles live across the last direction spill, 56-116 bytes of stack; there
                // the operand, prefetched into L2 at the start of the group, is loaded in the epilogue)
                if (EPI >= EPI_XPAY && u == 3 && active && sizeof(T) == 4) load_spinor(A.in2 + own, rowV, e0, qv);
                mbar_wait(&full[slot], use & 1);
                if (active) {
                    const vec* sp = reinterpret_cast<const vec*>(ring) + A.big_vecs + (size_t)(slot - 1) * A.small_vecs +
                                    (size_t)j * NCH * rowV;
                    const vec* lk = reinterpret_cast<const vec*>(ring) + A.big_vecs + (size_t)(slot - 1) * A.small_vecs +
                                    (size_t)RG * NCH * rowV + (size_t)j * lrowV;
                    if (u == 0)      dir_smem<T, RECON, 2, true, DAG>(sp, rowV, e0, lk, A.Lxh, xh, acc);
                    else if (u == 1) dir_smem<T, RECON, 2, false, DAG>(sp, rowV, e0, lk, A.Lxh, xh, acc);
                    else if (u == 2) dir_smem<T, RECON, 3, true, DAG>(sp, rowV, e0, lk, A.Lxh, xh, acc);
                    else             dir_smem<T, RECON, 3, false, DAG>(sp, rowV, e0, lk, A.Lxh, xh, acc);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[slot]);
            }
            ++q;
            // ---- epilogue and store
            if (active) {
                if (EPI >= EPI_XPAY) {
                    if (sizeof(T) == 8) load_spinor(A.in2 + own, rowV, e0, qv);
#pragma unroll
                    for (int k = 0; k < 12; ++k) {
                        acc[k].re = fma(A.b, acc[k].re, A.a * qv[k].re);
                        acc[k].im = fma(A.b, acc[k].im, A.a * qv[k].im);
                    }
                    if (EPI == EPI_OMEGA) {  // <t, s>, <t, t> with t = acc, s = qv
                        T s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
                        for (int k = 0; k < 12; ++k) {
                            s0 = fma(acc[k].re, qv[k].re, s0);  s0 = fma(acc[k].im, qv[k].im, s0);
                            s1 = fma(acc[k].re, qv[k].im, s1);  s1 = fma(-acc[k].im, qv[k].re, s1);
                            s2 = fma(acc[k].re, acc[k].re, s2); s2 = fma(acc[k].im, acc[k].im, s2);
                        }
                        dsum[0] += (double)s0; dsum[1] += (double)s1; dsum[2] += (double)s2;
                    }
                }
                if (EPI == EPI_SIGMA) {  // <r~, v> with v = acc
                    load_spinor(A.in3 + own, rowV, e0, qv);
                    T s0 = 0, s1 = 0;
#pragma unroll
                    for (int k = 0; k < 12; ++k) {
                        s0 = fma(qv[k].re, acc[k].re, s0);  s0 = fma(qv[k].im, acc[k].im, s0);
                        s1 = fma(qv[k].re, acc[k].im, s1);  s1 = fma(-qv[k].im, acc[k].re, s1);
                    }
                    dsum[0] += (double)s0; dsum[1] += (double)s1;
                }
                store_spinor(A.out + own, rowV, e0, acc);
            }
        }
    }
    if (EPI >= EPI_SIGMA) {
        // per-column sums of this CTA -> one partial per (column, value)
        constexpr int K = EPI == EPI_SIGMA ? 2 : 3;
        __syncthreads();  // every bulk copy has been consumed: the ring is free
        double* red = reinterpret_cast<double*>(ring);
        if (threadIdx.x < nct) {
#pragma unroll
            for (int k = 0; k < K; ++k) red[k * nct + threadIdx.x] = dsum[k];
        }
        __syncthreads();
        const uint32_t nwarps = blockDim.x >> 5;
        for (uint32_t item = warp; item < A.n * K; item += nwarps) {
            const uint32_t col = item / K, k = item - col * K;
            double v = 0.0;
            for (uint32_t ss = lane; ss < A.S; ss += 32) v += red[k * nct + ss * A.n + col];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) A.rb.partials[(size_t)item * gridDim.x + blockIdx.x] = v;
        }
        // With at most one CTA per SM there are few partials: the last CTA to get here adds them (fixed order) and
        // runs the scalar recurrence itself, so no finalize kernel follows this launch.
        double* tot = red + K * nct;   // n * K totals behind the per-thread sums, then the "last CTA" flag
        volatile uint32_t* is_last = reinterpret_cast<volatile uint32_t*>(tot + A.n * K);  // (no static shared memory: the
        __threadfence();                                                                    //  ring may take all 227 KB)
        __syncthreads();
        if (threadIdx.x == 0) *is_last = (atomicAdd(A.rb.ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
        __syncthreads();
        if (*is_last == 0u) return;
        __threadfence();
        for (uint32_t item = warp; item < A.n * K; item += nwarps) {
            const double* p = A.rb.partials + (size_t)item * gridDim.x;
            double v = 0.0;
            for (uint32_t g = lane; g < gridDim.x; g += 32) v += __ldcg(p + g);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) tot[item] = v;
        }
        __syncthreads();
        if (threadIdx.x < A.n)
            wdblas::finalize_column<EPI == EPI_SIGMA ? wdblas::K_SIGMA : wdblas::K_OMEGA>(A.rb.scal, (int)threadIdx.x, tot + threadIdx.x * K);
        if (threadIdx.x == 0) *A.rb.ticket = 0u;
    }
}

// ---- host side ----------------------------------------------------------------------------------------------
constexpr size_t kSmemMax = 227 * 1024;

struct Shape {
    uint32_t RG, S, threads, big_vecs, small_vecs, NS, NP;
    size_t smem;
};

// largest row group (a divisor of Ly) whose CTA fits the thread budget and whose ring fits shared memory
template <typename T, int RECON>
bool pick_shape(const wd_ctx* c, int n, int max_threads, Shape* sh) {
    const uint32_t Lxh = c->L[0] / 2, Ly = c->L[1];
    const uint32_t cap = c->opt[WD_OPT_HOP_ROWS] > 0 ? (uint32_t)c->opt[WD_OPT_HOP_ROWS] : Ly;
    for (uint32_t RG = Ly; RG >= 1; --RG) {
        if (Ly % RG || RG > cap) continue;
        const uint32_t S = RG * Lxh, rowV = Lxh * n;
        // consumer warps + a producer warp; a second one (it helps when groups are small and frequent: 146 against
        // 166 us at n = 12) only if the block stays within the thread budget, i.e. keeps its registers
        const uint32_t cthreads = ((S * n + 31) / 32) * 32;
        if ((int)cthreads + 32 > max_threads) continue;
        const uint32_t NP = (int)cthreads + 64 <= max_threads ? 2u : 1u;
        const uint32_t threads = cthreads + 32 * NP;
        const uint32_t lrowV = Lxh * RECON * (uint32_t)sizeof(T) / 16;
        const uint32_t big = ((RG + 2) * Vec<T>::NCH * rowV + 4 * RG * lrowV + 7) / 8 * 8;
        const uint32_t small = (RG * Vec<T>::NCH * rowV + RG * lrowV + 7) / 8 * 8;
        if (128 + ((size_t)big + 3 * (size_t)small) * 16 > kSmemMax) continue;
        uint32_t NS = 3;  // as many small slots as fit (deeper prefetch), at least 3
        while (NS < 7 && 128 + ((size_t)big + (NS + 1) * (size_t)small) * 16 <= kSmemMax) ++NS;
        const size_t smem = 128 + ((size_t)big + NS * (size_t)small) * 16;
        sh->NS = NS;
        sh->NP = NP;
        sh->RG = RG; sh->S = S; sh->threads = threads; sh->big_vecs = big; sh->small_vecs = small; sh->smem = smem;
        return true;
    }
    return false;
}

template <typename T, int RECON, bool DAG, int EPI, int MAXT>
int launch_one(wd_ctx* c, const TmaArgs<T>& A, const Shape& sh, unsigned G) {
    auto kern = hop_tma_kernel<T, RECON, DAG, EPI, MAXT>;
    WD_CUDA_CHECK(c, wd_ensure_smem_attr(c, (const void*)kern, (int)kSmemMax));
    kern<<<G, sh.threads, sh.smem, c->stream>>>(A);
    return WD_OK;
}

template <typename T, int RECON, int MAXT>
int launch_tma(wd_ctx* c, int dag, int n, int par, const wd_hop_ops& o, const T* U) {
    Shape sh;
    if (!pick_shape<T, RECON>(c, n, MAXT, &sh)) return 1;
    TmaArgs<T> A;
    A.in = (const typename Vec<T>::type*)o.in;
    A.out = (typename Vec<T>::type*)o.out;
    A.in2 = (const typename Vec<T>::type*)o.in2;
    A.in3 = (const typename Vec<T>::type*)o.in3;
    A.U = U;
    A.rb = wdblas::RedBuf{c->d_scal, c->d_partials, c->d_ticket};
    A.done = o.check_done ? c->d_scal + wdblas::G_DONE : nullptr;
    A.Lxh = c->L[0] / 2; A.Ly = c->L[1]; A.Lz = c->L[2]; A.Lt = c->L[3];
    A.Vh = (uint32_t)c->Vh; A.n = (uint32_t)n; A.par = (uint32_t)par; A.total = (uint32_t)(c->Vh * n);
    A.RG = sh.RG; A.S = sh.S;
    const uint32_t gy = A.Ly / sh.RG;
    A.groups = gy * A.Lz * A.Lt;
    A.g_first = c->bc == WD_BC_SF ? gy * A.Lz : 0;
    A.big_vecs = sh.big_vecs; A.small_vecs = sh.small_vecs; A.NS = sh.NS; A.NP = sh.NP;
    A.a = (T)o.a; A.b = (T)o.b;
    const uint32_t real = A.groups - A.g_first;
    const unsigned G = real < (uint32_t)c->n_sm ? real : (unsigned)c->n_sm;
    int rc;
#define WD_TMA_CASE(D, E) rc = launch_one<T, RECON, D, E, MAXT>(c, A, sh, G)
    if (dag) {
        if (o.epi == EPI_NONE) WD_TMA_CASE(true, EPI_NONE);
        else if (o.epi == EPI_XPAY) WD_TMA_CASE(true, EPI_XPAY);
        else if constexpr (sizeof(T) == 4) { if (o.epi == EPI_SIGMA) WD_TMA_CASE(true, EPI_SIGMA); else WD_TMA_CASE(true, EPI_OMEGA); }
        else return 1;
    } else {
        if (o.epi == EPI_NONE) WD_TMA_CASE(false, EPI_NONE);
        else if (o.epi == EPI_XPAY) WD_TMA_CASE(false, EPI_XPAY);
        else if constexpr (sizeof(T) == 4) { if (o.epi == EPI_SIGMA) WD_TMA_CASE(false, EPI_SIGMA); else WD_TMA_CASE(false, EPI_OMEGA); }
        else return 1;
    }
#undef WD_TMA_CASE
    if (rc) return rc;
    return WD_OK;
}

}  // namespace

// Would wd_hop_tma_launch serve plain operands of this precision and link form? (same conditions, nothing launched)
bool wd_hop_tma_serves(const wd_ctx* c, int prec, int recon, int n) {
    if (c->order != WD_ORDER_LINEAR || c->RB != (uint32_t)(c->L[0] / 2)) return false;
    Shape sh;
    if (prec == WD_F64) return recon == WD_LINK18 ? pick_shape<double, 18>(c, n, 384, &sh) : pick_shape<double, 12>(c, n, 384, &sh);
    return recon == WD_LINK18 ? pick_shape<float, 18>(c, n, 512, &sh) : pick_shape<float, 12>(c, n, 512, &sh);
}

// Returns WD_OK if launched, a positive value if this lattice / option set is not served by the staged kernel
// (tiled site order, odd Lx/2 with 18-real fp32 links, nothing fits): the caller then uses wd_hop.cu's kernel.
int wd_hop_tma_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o) {
    if (c->order != WD_ORDER_LINEAR || c->RB != (uint32_t)(c->L[0] / 2)) return 1;  // needs the row-major layout
    int rc;
    if (prec == WD_F64) {
        if (recon == WD_LINK18) rc = launch_tma<double, 18, 384>(c, dag, n, par, o, c->d_U64[0]);
        else                    rc = launch_tma<double, 12, 384>(c, dag, n, par, o, c->d_U64[1]);
    } else {
        if (recon == WD_LINK18) rc = launch_tma<float, 18, 512>(c, dag, n, par, o, c->d_U32[0]);
        else                    rc = launch_tma<float, 12, 512>(c, dag, n, par, o, c->d_U32[1]);
    }
    return rc;
}
