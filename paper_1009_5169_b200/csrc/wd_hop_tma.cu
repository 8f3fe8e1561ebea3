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
// Measured (B200, 24^4, fp32, 12-real links, L2-cold): bit-identical results to the register kernel; 75.9 us
// against 70.5 us at n_rhs = 5, 172 us against 194 us at n_rhs = 12.  With the consumers' arithmetic switched off
// the producer alone needs 49 us: each bulk copy costs about 85 ns of issue/latency, and in the chunk-major native
// layout a group needs about 60 copies of 1-4 KB (one per spinor chunk and link chunk).  So this form is the
// opt-in choice (WD_OPT_HOP_IMPL = 1; it wins from n_rhs ~ 12 up) until the native layout is row-major, which
// would bring a group down to ~15 copies; that layout change is listed under "next" in DESIGN.md.
//
// A note for whoever touches the producer: keep its copy loops rolled.  Fully unrolled for fp64 (12 chunks) ptxas
// ran out of uniform registers and emitted R2UR.FILL spills around the UBLKCP instructions; that build raised
// "illegal memory access" on every fp64 launch although every address and size checked out.
//
// Geometry (linear site order only): a half-lattice index is h = xh + Lxh*(y + Ly*(z + Lz*t)), xh = x/2.
// A "row" is the Lxh sites of fixed (y,z,t); neighbours in +-y, +-z, +-t of a row are the row with the
// same xh at the shifted (y,z,t); neighbours in +-x are in the row with the same (y,z,t) of the other
// parity at xh or xh+-1 (which one depends on the parity of y+z+t+par).  So no neighbour table is read.
// Work item = a group of RG consecutive rows in y (S = RG*Lxh sites, S*n consumer threads).  Per group the
// producer issues 5 units:  XY (input rows y0-1 .. y0+RG, links x+ x- y+ y-), Z+, Z-, T+, T- (RG input rows
// and one link array each).  Ring: one big slot for XY units and three small slots for the others.
#include "wd_blas.cuh"
#include "wd_su3.cuh"

using namespace wdk;

namespace {

enum { EPI_NONE = 0, EPI_XPAY = 1, EPI_SIGMA = 2, EPI_OMEGA = 3 };

// ---- mbarrier / bulk-copy PTX ---------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}
// global -> shared bulk copy, completion counted in bytes on `bar` (sizes and addresses multiples of 16)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}


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
    T a, b;
};

template <typename T, int RECON> struct LinkShape;
template <> struct LinkShape<float, 12> { enum { CH16 = 3, TAIL8 = 0 }; };
template <> struct LinkShape<float, 18> { enum { CH16 = 4, TAIL8 = 1 }; };   // + one float2 chunk
template <> struct LinkShape<double, 12> { enum { CH16 = 6, TAIL8 = 0 }; };
template <> struct LinkShape<double, 18> { enum { CH16 = 9, TAIL8 = 0 }; };

// 16-byte units of one staged link array of S sites
template <typename T, int RECON>
__host__ __device__ constexpr uint32_t link_vecs(uint32_t S) {
    return LinkShape<T, RECON>::CH16 * S + (LinkShape<T, RECON>::TAIL8 ? (S + 1) / 2 : 0);
}

__device__ __forceinline__ uint32_t wrap_inc(uint32_t v, uint32_t L) { return v + 1 == L ? 0u : v + 1; }
__device__ __forceinline__ uint32_t wrap_dec(uint32_t v, uint32_t L) { return v == 0 ? L - 1 : v - 1; }

// ---- producer side ------------------------------------------------------------------------------------
// The producer WARP issues the copies of a unit lane-parallel: copy number idx -> (dst, src, bytes) is pure index
// arithmetic, every lane works out its own and the hardware serialises only the UBLKCP issue itself.  (One thread
// issuing all ~70 copies of a group took longer than the consumers' arithmetic on that group.)
//
// One copy = (dst, src, bytes).  Every lane fills in its own descriptor with selects and all lanes meet at ONE
// bulk_g2s call site, so the hardware-serialised part is just the UBLKCP issue.
struct CopyDesc {
    char* dst;
    const char* src;
    uint32_t bytes;  // 0 = nothing to copy
};

// piece of a staged link array: `count` consecutive sites from half-lattice index hsrc of link block (mu, q) go to
// site offset `off` of the array at L; copy cc < CH16 is 16-byte chunk cc, copy CH16 the float2 tail (fp32 R=18)
template <typename T, int RECON>
__device__ __forceinline__ CopyDesc link_desc(const TmaArgs<T>& A, char* L, int mu, uint32_t q, uint32_t hsrc, uint32_t count,
                                              uint32_t off, uint32_t cc) {
    constexpr uint32_t CH16 = LinkShape<T, RECON>::CH16;
    const char* blk = reinterpret_cast<const char*>(A.U + (size_t)(mu * 2 + q) * RECON * A.Vh);
    CopyDesc d;
    if (cc < CH16) {
        d.dst = L + ((size_t)cc * A.S + off) * 16;
        d.src = blk + ((size_t)cc * A.Vh + hsrc) * 16;
        d.bytes = count * 16;
    } else {
        d.dst = L + (size_t)CH16 * A.S * 16 + (size_t)off * 8;
        d.src = blk + ((size_t)16 * A.Vh + 2 * (size_t)hsrc) * 4;
        d.bytes = count * 8;
    }
    return d;
}

template <typename T, int RECON>
__device__ void produce_group(const TmaArgs<T>& A, uint32_t lane, uint32_t y0, uint32_t z, uint32_t t, uint32_t q, char* ring,
                              uint64_t* full, uint64_t* empty) {
    constexpr uint32_t NCH = Vec<T>::NCH;
    constexpr uint32_t CHT = LinkShape<T, RECON>::CH16 + LinkShape<T, RECON>::TAIL8;                 // copies per link piece
    constexpr uint32_t LB = LinkShape<T, RECON>::CH16 * 16 + LinkShape<T, RECON>::TAIL8 * 8;         // bytes per link
    const uint32_t rowV = A.Lxh * A.n, rowB = rowV * 16, RG = A.RG, S = A.S;
    const uint32_t zt = z + A.Lz * t;
    const uint32_t row0 = y0 + A.Ly * zt;
    const uint32_t h0 = row0 * A.Lxh;
    const char* in = reinterpret_cast<const char*>(A.in);
    const size_t chB = (size_t)A.total * 16;  // bytes per spinor chunk
    // ---- XY unit -> big slot (use q)
    {
        mbar_wait(&empty[0], (q & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&full[0], NCH * (RG + 2) * rowB + 4 * S * LB);
        __syncwarp();
        char* B = ring;
        char* L = B + (size_t)NCH * (RG + 2) * rowB;
        const size_t LVB = (size_t)link_vecs<T, RECON>(S) * 16;
        const bool lo = y0 == 0, hi = y0 + RG == A.Ly;   // the halo row below / above wraps around in y
        const uint32_t rm = (lo ? A.Ly - 1 : y0 - 1) + A.Ly * zt;
        const uint32_t rp = (hi ? 0 : y0 + RG) + A.Ly * zt;
        for (uint32_t idx = lane; idx < 3 * NCH + 5 * CHT; idx += 32) {
            CopyDesc d;
            if (idx < 3 * NCH) {
                // input rows of chunk c: segment 1 = rows y0 .. y0+RG-1 together with whichever halo rows are contiguous
                // with them; segments 0 / 2 = the halo row below / above only when it wraps
                const uint32_t c = idx / 3, seg = idx - 3 * c;
                char* dc = B + (size_t)c * (RG + 2) * rowB;
                const char* sc = in + c * chB;
                if (seg == 1) {
                    const uint32_t first = lo ? 1u : 0u, nrows = RG + (lo ? 0u : 1u) + (hi ? 0u : 1u);
                    d.dst = dc + (size_t)first * rowB;
                    d.src = sc + (size_t)(row0 - (lo ? 0u : 1u)) * rowB;
                    d.bytes = nrows * rowB;
                } else if (seg == 0) {
                    d.dst = dc; d.src = sc + (size_t)rm * rowB; d.bytes = lo ? rowB : 0u;
                } else {
                    d.dst = dc + (size_t)(RG + 1) * rowB; d.src = sc + (size_t)rp * rowB; d.bytes = hi ? rowB : 0u;
                }
            } else {
                const uint32_t k = idx - 3 * NCH, piece = k / CHT, cc = k - piece * CHT;
                // pieces: x+ U_x(x) | x- U_x on the same rows of the other parity | y+ U_y(x) | y- row y0-1 | y- rows y0 ..
                const uint32_t arr = piece < 3 ? piece : 3u;
                const int mu = piece < 2 ? 0 : 1;
                const uint32_t qq = (piece == 0 || piece == 2) ? A.par : 1 - A.par;
                const uint32_t hsrc = piece == 3 ? rm * A.Lxh : h0;
                const uint32_t count = piece == 3 ? A.Lxh : (piece == 4 ? S - A.Lxh : S);
                const uint32_t off = piece == 4 ? A.Lxh : 0u;
                d = link_desc<T, RECON>(A, L + arr * LVB, mu, qq, hsrc, count, off, cc);
            }
            if (d.bytes) bulk_g2s(d.dst, d.src, d.bytes, &full[0]);
        }
    }
    // ---- Z+, Z-, T+, T- units -> small slots
    const size_t bigB = (size_t)A.big_vecs * 16, smallB = (size_t)A.small_vecs * 16;
#pragma unroll 1
    for (uint32_t u = 0; u < 4; ++u) {
        const uint32_t m = 4 * q + u, slot = 1 + m % 3, use = m / 3;
        mbar_wait(&empty[slot], (use & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&full[slot], NCH * RG * rowB + S * LB);
        __syncwarp();
        char* B = ring + bigB + (size_t)(slot - 1) * smallB;
        uint32_t zz = z, tt = t;
        if (u == 0) zz = wrap_inc(z, A.Lz);
        else if (u == 1) zz = wrap_dec(z, A.Lz);
        else if (u == 2) tt = wrap_inc(t, A.Lt);
        else tt = wrap_dec(t, A.Lt);
        const uint32_t rn = y0 + A.Ly * (zz + A.Lz * tt);
        const bool fwd = (u & 1) == 0;
        for (uint32_t idx = lane; idx < NCH + CHT; idx += 32) {
            CopyDesc d;
            if (idx < NCH) {
                d.dst = B + (size_t)idx * RG * rowB; d.src = in + idx * chB + (size_t)rn * rowB; d.bytes = RG * rowB;
            } else {
                d = link_desc<T, RECON>(A, B + (size_t)NCH * RG * rowB, 2 + (u >> 1), fwd ? A.par : 1 - A.par,
                                        fwd ? h0 : rn * A.Lxh, S, 0, idx - NCH);
            }
            if (d.bytes) bulk_g2s(d.dst, d.src, d.bytes, &full[slot]);
        }
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
// grid = min(groups, SMs) persistent CTAs; block = consumer warps (S*n threads, rounded up) + 1 producer warp.
// dynamic smem: 128 bytes of mbarriers, then the ring: [big slot][3 small slots].
template <typename T, int RECON, bool DAG, int EPI, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) hop_tma_kernel(const TmaArgs<T> A) {
    typedef typename Vec<T>::type vec;
    if (A.done != nullptr && *A.done != 0.0) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* empty = full + 4;
    char* ring = reinterpret_cast<char*>(smem) + 128;
    const uint32_t nct = A.S * A.n;            // consumer threads
    const uint32_t ncw = (nct + 31) >> 5;      // consumer warps
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < 4; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], ncw); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t gy = A.Ly / A.RG;
    [[maybe_unused]] double dsum[3] = {0.0, 0.0, 0.0};

    if (warp == ncw) {
        // ================= producer warp: issues every bulk copy of this CTA's groups ======================
        uint32_t q = 0;
        for (uint32_t g = A.g_first + blockIdx.x; g < A.groups; g += gridDim.x) {
            const uint32_t yg = g % gy, zt = g / gy, z = zt % A.Lz, t = zt / A.Lz;
            produce_group<T, RECON>(A, lane, yg * A.RG, z, t, q, ring, full, empty);
            ++q;
        }
    } else {
        // ================= consumers: thread i = (site s of the group, column r) =========================
        const uint32_t i = threadIdx.x;
        const bool active = i < nct;
        const uint32_t s = i / A.n, r = i - s * A.n;
        const uint32_t j = s / A.Lxh, xh = s - j * A.Lxh;
        const uint32_t rowV = A.Lxh * A.n, RG = A.RG, S = A.S;
        const vec* bigS = reinterpret_cast<const vec*>(ring);
        const vec* bigL = bigS + (size_t)Vec<T>::NCH * (RG + 2) * rowV;
        const uint32_t LV = link_vecs<T, RECON>(S);
        const uint32_t smallLoff = Vec<T>::NCH * RG * rowV;
        uint32_t q = 0;
        if (active) {  // SF: the stored t = 0 slice stays zero
            cx<T> zero[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) { zero[k].re = 0; zero[k].im = 0; }
            for (uint32_t g = blockIdx.x; g < A.g_first; g += gridDim.x) store_spinor(A.out, A.total, g * S * A.n + i, zero);
        }
        for (uint32_t g = A.g_first + blockIdx.x; g < A.groups; g += gridDim.x) {
            const uint32_t yg = g % gy, zt = g / gy, z = zt % A.Lz, t = zt / A.Lz;
            const uint32_t y0 = yg * RG;
            const uint32_t oidx = (y0 + A.Ly * zt) * rowV + i;  // h0 * n + i
            cx<T> acc[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) { acc[k].re = 0; acc[k].im = 0; }
            // ---- XY unit
            mbar_wait(&full[0], q & 1);
            if (active) {
                const uint32_t b = (y0 + j + z + t + A.par) & 1;
                const uint32_t xp = b ? wrap_inc(xh, A.Lxh) : xh;   // xh of the +x neighbour
                const uint32_t xm = b ? xh : wrap_dec(xh, A.Lxh);   // xh of the -x neighbour
                const uint32_t st = (RG + 2) * rowV;
                dir_smem<T, RECON, 0, true, DAG>(bigS, st, (j + 1) * rowV + xp * A.n + r, bigL, S, s, acc);
                dir_smem<T, RECON, 0, false, DAG>(bigS, st, (j + 1) * rowV + xm * A.n + r, bigL + LV, S, j * A.Lxh + xm, acc);
                dir_smem<T, RECON, 1, true, DAG>(bigS, st, (j + 2) * rowV + xh * A.n + r, bigL + 2 * LV, S, s, acc);
                dir_smem<T, RECON, 1, false, DAG>(bigS, st, j * rowV + xh * A.n + r, bigL + 3 * LV, S, s, acc);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[0]);
            // ---- Z+, Z-, T+, T- units
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t m = 4 * q + u, slot = 1 + m % 3, use = m / 3;
                mbar_wait(&full[slot], use & 1);
                if (active) {
                    const vec* sp = reinterpret_cast<const vec*>(ring) + A.big_vecs + (size_t)(slot - 1) * A.small_vecs;
                    if (u == 0)      dir_smem<T, RECON, 2, true, DAG>(sp, S * A.n, i, sp + smallLoff, S, s, acc);
                    else if (u == 1) dir_smem<T, RECON, 2, false, DAG>(sp, S * A.n, i, sp + smallLoff, S, s, acc);
                    else if (u == 2) dir_smem<T, RECON, 3, true, DAG>(sp, S * A.n, i, sp + smallLoff, S, s, acc);
                    else             dir_smem<T, RECON, 3, false, DAG>(sp, S * A.n, i, sp + smallLoff, S, s, acc);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[slot]);
            }
            ++q;
            // ---- epilogue and store
            if (active) {
                if (EPI >= EPI_XPAY) {
                    cx<T> qv[12];
                    load_spinor(A.in2, A.total, oidx, qv);
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
                    cx<T> qv[12];
                    load_spinor(A.in3, A.total, oidx, qv);
                    T s0 = 0, s1 = 0;
#pragma unroll
                    for (int k = 0; k < 12; ++k) {
                        s0 = fma(qv[k].re, acc[k].re, s0);  s0 = fma(qv[k].im, acc[k].im, s0);
                        s1 = fma(qv[k].re, acc[k].im, s1);  s1 = fma(-qv[k].im, acc[k].re, s1);
                    }
                    dsum[0] += (double)s0; dsum[1] += (double)s1;
                }
                store_spinor(A.out, A.total, oidx, acc);
            }
        }
    }
    if (EPI >= EPI_SIGMA) {
        // per-column sums of this CTA -> one partial per (column, value); finalize_partials_kernel follows
        constexpr int K = EPI == EPI_SIGMA ? 2 : 3;
        __syncthreads();  // every bulk copy has been consumed: the ring is free
        double* red = reinterpret_cast<double*>(ring);
        if (warp != ncw && threadIdx.x < nct) {
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
    }
}

// ---- host side ----------------------------------------------------------------------------------------------
constexpr size_t kSmemMax = 227 * 1024;

struct Shape {
    uint32_t RG, S, threads, big_vecs, small_vecs;
    size_t smem;
};

// largest row group (a divisor of Ly) whose CTA fits the thread budget and whose ring fits shared memory
template <typename T, int RECON>
bool pick_shape(const wd_ctx* c, int n, int max_threads, Shape* sh) {
    const uint32_t Lxh = c->L[0] / 2, Ly = c->L[1];
    for (uint32_t RG = Ly; RG >= 1; --RG) {
        if (Ly % RG) continue;
        const uint32_t S = RG * Lxh, rowV = Lxh * n;
        const uint32_t threads = ((S * n + 31) / 32) * 32 + 32;
        if ((int)threads > max_threads) continue;
        const uint32_t LV = link_vecs<T, RECON>(S);
        const uint32_t big = (Vec<T>::NCH * (RG + 2) * rowV + 4 * LV + 7) / 8 * 8;
        const uint32_t small = (Vec<T>::NCH * RG * rowV + LV + 7) / 8 * 8;
        const size_t smem = 128 + ((size_t)big + 3 * (size_t)small) * 16;
        if (smem > kSmemMax) continue;
        sh->RG = RG; sh->S = S; sh->threads = threads; sh->big_vecs = big; sh->small_vecs = small; sh->smem = smem;
        return true;
    }
    return false;
}

template <typename T, int RECON, bool DAG, int EPI, int MAXT>
int launch_one(wd_ctx* c, const TmaArgs<T>& A, const Shape& sh, unsigned G) {
    static bool attr_set = false;
    auto kern = hop_tma_kernel<T, RECON, DAG, EPI, MAXT>;
    if (!attr_set) {
        WD_CUDA_CHECK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));
        attr_set = true;
    }
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
    A.big_vecs = sh.big_vecs; A.small_vecs = sh.small_vecs;
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
    if (o.epi == EPI_SIGMA)
        wdblas::finalize_partials_kernel<2, wdblas::K_SIGMA><<<2 * n, 256, 0, c->stream>>>(n, G, A.rb, c->d_totals);
    else if (o.epi == EPI_OMEGA)
        wdblas::finalize_partials_kernel<3, wdblas::K_OMEGA><<<3 * n, 256, 0, c->stream>>>(n, G, A.rb, c->d_totals);
    if (o.epi >= EPI_SIGMA) c->launches++;
    return WD_OK;
}

}  // namespace

// Returns WD_OK if launched, a positive value if this lattice / option set is not served by the staged kernel
// (tiled site order, odd Lx/2 with 18-real fp32 links, nothing fits): the caller then uses wd_hop.cu's kernel.
int wd_hop_tma_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o) {
    if (c->order != WD_ORDER_LINEAR) return 1;
    const uint32_t Lxh = c->L[0] / 2;
    if (prec == WD_F32 && recon == WD_LINK18 && (Lxh & 1)) return 1;  // the float2 chunk needs 16-byte pieces
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
