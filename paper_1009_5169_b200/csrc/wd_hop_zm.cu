// wd_hop_zm.cu -- the multi-RHS Wilson hopping kernel (hot-path step a2), "z-march" form:
// persistent CTAs that walk along z with a sliding window of three lattice planes resident in shared memory.
//
// Why: the first staged kernel (wd_hop_tma.cu) re-stages the z+-1 and t+-1 neighbours of every group of 8 rows,
// 42 input rows per 8 output rows = 5.25 x the input spinor through the L2 -> SM path (ncu r01e: 524 MB per launch
// against 223 MB algorithmic; "producers alone" 43 us = the L2 read ceiling), and it consumes a unit in 0.35 us
// that takes >= 1 us to arrive, with a ring that is one group deep.  Here a CTA owns a "column" (RG consecutive
// rows in y at fixed t) and marches z = z0, z0+1, ...: the centre plane of one step is the z- plane of the next
// and its z+ plane becomes the centre, so per step only ONE new plane (RG rows), the two y-halo rows and the
// t+-1 rows (2 RG) are copied: (3 RG + 2) / RG = 3.33 x at RG = 6 instead of 5.25 x.  Every buffer is released
// as soon as its last direction has been consumed (order t+, t-, z-, y-, y+, x-, x+, z+) and refilled for the
// next step while the rest of this step computes, so each copy has about one step time (~2 us) to land.
//
// Geometry (linear site order, row-major native layout RB = Lx/2, as wd_hop_tma.cu): row = (y, z, t), Lxh sites.
// Work: steps s = (column c, z), c = yb + gy * (t - t0), z fastest, S = gy (Lt - t0) Lz of them (t0 = 1 with
// Schroedinger-functional boundaries: the stored t = 0 slice stays zero and is only ever read as a neighbour),
// cut into chunks of `chunk` consecutive steps; CTA b takes chunks b, b + G, ...  When a chunk crosses into the
// next column the window restarts (three planes instead of one: a bubble of one copy latency).
//
// Shared memory (fp32, 24^4, n = 5, RG = 6, 18-real links: 225.9 KB): 3 planes x RG rows | T+ RG rows | T- RG rows
// | 2 halo rows | links: 8 blocks of RG link rows in consumption order.  Units and their barriers:
//   U1 {T+ rows, link t+}  U2 {T- rows, link t-}  U3 {link z-}  U4 {halo rows, links y-, y+}  U5 {links x-, x+, z+}
//   W[j % 3] plane with sequence number j (consecutive z of a column; +3 at a column switch).
// Four producer warps issue the cp.async.bulk copies; consumer thread = (site of the step, column r),
// r fastest: conflict-free 128-bit shared-memory reads, results bit for bit those of the register kernel
// (wd_hop.cu accumulates the directions in the same order).
#include "wd_blas.cuh"
#include "wd_f2.cuh"
#include "wd_h16.cuh"
#include "wd_su3.cuh"
#include "wd_tma.cuh"

using namespace wdk;
using namespace wdtma;

namespace {
#ifndef WD_ZM_ABLATE
#define WD_ZM_ABLATE 0   // measurement builds only (build.py WD_NVCC_DEFINES, profiles/r02_hop_ablations.md): 1 = consumers skip the arithmetic, 2 = no copies, no waits
#endif
#if WD_ZM_ABLATE == 2
#define mbar_wait(b, p) ((void)0)
#define mbar_wait_relaxed(b, p) ((void)0)
#define bulk_g2s(d, s, n, b) ((void)0)
#define mbar_expect_tx(b, n) ((void)0)
#endif

// EPI_OMEGA_RHO (plain fp32 operands only): EPI_OMEGA plus <in3, in2> and <in3, out>, i.e. <rt,s> and <rt,t> for the merged-update
// schedule of the solver (7 sums per column)
enum { EPI_NONE = 0, EPI_XPAY = 1, EPI_SIGMA = 2, EPI_OMEGA = 3, EPI_OMEGA_RHO = 4 };
enum { U_TP = 0, U_TM = 1, U_ZM = 2, U_Y = 3, U_XZ = 4, NUNIT = 5 };
// link blocks in shared memory, in consumption order
enum { LK_TP = 0, LK_TM = 1, LK_ZM = 2, LK_YM = 3, LK_YP = 4, LK_XM = 5, LK_XP = 6, LK_ZP = 7 };

template <typename T>
struct ZmArgs {
    const typename Vec<T>::type* in;
    typename Vec<T>::type* out;
    const typename Vec<T>::type* in2;
    const typename Vec<T>::type* in3;
    const T* U;
    wdblas::RedBuf rb;
    const double* done;
    uint32_t Lxh, Ly, Lz, Lt;
    uint32_t Vh, n, par;
    uint32_t RG, S;          // rows per step, sites per step = RG * Lxh
    uint32_t gy;             // Ly / RG
    uint32_t t0;             // first dynamical time slice
    uint32_t steps;          // gy * (Lt - t0) * Lz
    uint32_t chunk;          // steps per chunk; CTA b takes chunks b, b + G, ...
    uint32_t zero_rows;      // rows of the frozen t = 0 slice to clear (SF), else 0
    T a, b;
};

__device__ __forceinline__ uint32_t winc(uint32_t v, uint32_t L) { return v + 1 == L ? 0u : v + 1; }
__device__ __forceinline__ uint32_t wdec(uint32_t v, uint32_t L) { return v == 0 ? L - 1 : v - 1; }

// Step sequence of a CTA: chunks b, b + G, ... of `chunk` consecutive steps each.  NO_STEP ends it.
constexpr uint32_t NO_STEP = 0xffffffffu;
__device__ __forceinline__ uint32_t next_step(uint32_t s, uint32_t chunk, uint32_t steps) {
    if ((s + 1) % chunk != 0 && s + 1 < steps) return s + 1;
    const uint32_t f = (s / chunk + gridDim.x) * chunk;
    return f < steps ? f : NO_STEP;
}
// does step s2 continue the z-march of step s1 (same column, next z)?  Then the window slides by one plane.
__device__ __forceinline__ bool continues(uint32_t s1, uint32_t s2, uint32_t Lz) { return s2 == s1 + 1 && s2 / Lz == s1 / Lz; }

// ---- shared-memory operand reads ---------------------------------------------------------------------------
__device__ __forceinline__ void lds_spinor(const float4* __restrict__ sp, uint32_t stride, uint32_t e, cx<float> (&psi)[12]) {
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float4 v = sp[c * stride + e];
        psi[2 * c].re = v.x; psi[2 * c].im = v.y; psi[2 * c + 1].re = v.z; psi[2 * c + 1].im = v.w;
    }
}
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

template <typename T, int RECON, int ST, int MU, bool FWD, bool DAG, bool FIRST = false>
__device__ __forceinline__ void dir_smem(const typename Vec<T>::type* sp, uint32_t stride, uint32_t e,
                                         const typename Vec<T>::type* L, uint32_t S, uint32_t site, cx<T> (&acc)[12]) {
    if (WD_ZM_ABLATE == 1) {
        if (FIRST) {
#pragma unroll
            for (int q = 0; q < 12; ++q) { acc[q].re = 0; acc[q].im = 0; }
        }
        return;
    }
    constexpr int SIGMA = (FWD ? 1 : -1) * (DAG ? -1 : 1);
    cx<T> psi[12], hs[6], chi[6], u[9];
    [[maybe_unused]] T scale = 1;
    if (ST) scale = wdh::h16_load_raw(sp, stride, e, psi); else lds_spinor(sp, stride, e, psi);
    lds_link<RECON>(L, S, site, u);
    if (RECON == 12) rebuild_row3(u);
    project<MU, SIGMA>(psi, hs);
    su3_mul<!FWD>(u, hs, chi);
    if (ST) {
#pragma unroll
        for (int q = 0; q < 6; ++q) { chi[q].re *= scale; chi[q].im *= scale; }
    }
    accumulate<MU, SIGMA, FIRST>(acc, chi);
}

// ---- the same for two sites per thread (ST = 2: P32 operands, wd_f2.cuh) ---------------------------------------
// The operands of one direction: the neighbour pair's spinor and the link, as loaded (12-real links before the rebuild).
// The consumers keep TWO of these: the loads of direction d + 1 are issued before the arithmetic of direction d, so that
// with six consumer warps per SM the shared-memory pipe and the FMA pipe work at the same time.
struct PairOps {
    wdp::cx2 psi[12];
    wdp::cx2 u[9];
};
// sp: spinor row in shared memory, cs = H * n elements per complex, e = element of the neighbour pair; L: link row,
// lp = pair whose link is used.
template <int RECON>
__device__ __forceinline__ void pair_load(PairOps& o, const ulonglong2* sp, uint32_t cs, uint32_t e, const ulonglong2* L, uint32_t H, uint32_t lp) {
    if (WD_ZM_ABLATE == 1) return;
    wdp::ld_spinor(sp, cs, e, o.psi);
    wdp::ld_link_raw<RECON>(L, H, lp, o.u);
}
// SWAP (x hops only): the neighbour pair has its lanes exchanged -- the forward hop exchanges the projected half spinor
// (the link is the output pair's own), the backward hop multiplies in the neighbour's lane order (its link sits with it)
// and exchanges the result.
template <int RECON, int MU, bool FWD, bool DAG, bool FIRST = false, bool SWAP = false>
__device__ __forceinline__ void pair_compute(PairOps& o, wdp::cx2 (&acc)[12], bool swp = false) {
    if (WD_ZM_ABLATE == 1) {
        if (FIRST) {
#pragma unroll
            for (int q = 0; q < 12; ++q) { acc[q].re = wdp::zero2(); acc[q].im = wdp::zero2(); }
        }
        return;
    }
    constexpr int SIGMA = (FWD ? 1 : -1) * (DAG ? -1 : 1);
    wdp::cx2 hs[6], chi[6];
    wdp::finish_link<RECON>(o.u);
    wdp::project<MU, SIGMA>(o.psi, hs);
    if (SWAP && FWD) {
#pragma unroll
        for (int q = 0; q < 6; ++q) { hs[q].re = wdp::swap_if(swp, hs[q].re); hs[q].im = wdp::swap_if(swp, hs[q].im); }
    }
    wdp::su3_mul<!FWD>(o.u, hs, chi);
    if (SWAP && !FWD) {
#pragma unroll
        for (int q = 0; q < 6; ++q) { chi[q].re = wdp::swap_if(swp, chi[q].re); chi[q].im = wdp::swap_if(swp, chi[q].im); }
    }
    wdp::accumulate<MU, SIGMA, FIRST>(acc, chi);
}

// ---- the kernel -------------------------------------------------------------------------------------------
// block = consumer warps (S * n threads, rounded up) + four producer warps; grid = min(steps, SMs).
// dynamic smem: 128 B of mbarriers | planes 3 x RG rows | T+ | T- | halo 2 rows | links 8 x RG link rows
// LXH, NR, RGT: Lx/2, n_rhs and rows per step as compile-time constants (0 = taken from the arguments).  With all
// three fixed every shared-memory operand address is one per-thread base register plus an immediate; with run-time
// strides the kernel spent 220 integer instructions per step and ~40 registers on addresses (ncu r02b).
// ST = 1: spinor blocks (in, out, in2, in3) are in the 16-bit storage format of wd_h16.cuh (arithmetic stays fp32).
template <typename T, int RECON, bool DAG, int EPI, int MAXT, int LXH, int NR, int RGT, int ST>
__global__ void __launch_bounds__(MAXT, 1) hop_zm_kernel(const ZmArgs<T> A) {
    typedef typename Vec<T>::type vec;
    constexpr uint32_t NCH = Vec<T>::NCH;
    if (A.done != nullptr && *A.done != 0.0) return;
    const uint32_t Lxh = LXH ? (uint32_t)LXH : A.Lxh, nr = NR ? (uint32_t)NR : A.n;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full_u = reinterpret_cast<uint64_t*>(smem);   // [5]
    uint64_t* empty_u = full_u + NUNIT;                      // [5]
    uint64_t* full_w = empty_u + NUNIT;                      // [3]
    uint64_t* empty_w = full_w + 3;                          // [3]
    const uint32_t RG = RGT ? (uint32_t)RGT : A.RG, rowV = Lxh * nr;
    const uint32_t rowS = ST == 1 ? wdh::h16_row_vecs(rowV) : NCH * rowV;   // 16-byte units of one spinor row (all chunks)
    const uint32_t SW = ST == 2 ? Lxh / 2 : Lxh;                            // thread-sites per row (ST = 2: site pairs)
    const uint32_t rowB = rowS * 16;                                     // bytes of one spinor row
    const uint32_t lrowB = Lxh * RECON * (uint32_t)sizeof(T);            // bytes of one row of one link array
    char* const base = reinterpret_cast<char*>(smem) + 128;
    char* const planes = base;
    char* const tp = planes + (size_t)3 * RG * rowB;
    char* const tm = tp + (size_t)RG * rowB;
    char* const halo = tm + (size_t)RG * rowB;
    char* const links = halo + (size_t)2 * rowB;
    const uint32_t nct = RG * SW * nr, ncw = (nct + 31) >> 5;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (uint32_t u = 0; u < NUNIT; ++u) { mbar_init(&full_u[u], 1); mbar_init(&empty_u[u], ncw); }
        for (uint32_t w = 0; w < 3; ++w) { mbar_init(&full_w[w], 1); mbar_init(&empty_w[w], ncw); }
        mbar_fence_init();
    }
    __syncthreads();
    const uint32_t s_first = blockIdx.x * A.chunk;   // < steps: the grid has at most ceil(steps / chunk) CTAs
    [[maybe_unused]] double dsum[EPI == EPI_OMEGA_RHO ? 7 : 3] = {};

    if (ST == 2 && warp >= ncw) {
        // ================= producer warps, P32 form: TWO warps (the consumers, two sites per thread with the next
        // direction's operands in flight, need ~250 registers: 256 threads per CTA).  A thread can start a bulk copy
        // only every ~280 ns, so every copy of a step has a lane of its own; the waits follow the order in which the
        // consumers release the buffers.
        //   P0: U1 {T+ rows, link t+}, U2 {T- rows, link t-}, U3 {link z-}, window planes      P1: U4, U5
        const uint32_t role = warp - ncw;
        const char* in = reinterpret_cast<const char*>(A.in);
        const char* U = reinterpret_cast<const char*>(A.U);
        const size_t ublk = (size_t)RECON * A.Vh * sizeof(T);
        uint32_t issued = 0, a = 0, prev = NO_STEP;
        for (uint32_t s = s_first, k = 0; s != NO_STEP; prev = s, s = next_step(s, A.chunk, A.steps), ++k) {
            const uint32_t col = s / A.Lz, z = s - col * A.Lz;
            const uint32_t yb = col % A.gy, t = A.t0 + col / A.gy, y0 = yb * RG;
            if (k > 0) a += continues(prev, s, A.Lz) ? 1u : 3u;
            const uint32_t eph = (k & 1) ^ 1;
            const uint32_t row0 = y0 + A.Ly * (z + A.Lz * t);
            if (role == 0) {
                const uint32_t rtp = y0 + A.Ly * (z + A.Lz * winc(t, A.Lt));
                const uint32_t rtm = y0 + A.Ly * (z + A.Lz * wdec(t, A.Lt));
                const uint32_t rzm = y0 + A.Ly * (wdec(z, A.Lz) + A.Lz * t);
                mbar_wait_relaxed(&empty_u[U_TP], eph);
                if (lane == 0) mbar_expect_tx(&full_u[U_TP], RG * (rowB + lrowB));
                __syncwarp();
                if (lane == 0) bulk_g2s(tp, in + (size_t)rtp * rowB, RG * rowB, &full_u[U_TP]);
                else if (lane == 1) bulk_g2s(links + (size_t)LK_TP * RG * lrowB, U + (size_t)(6 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_TP]);
                mbar_wait_relaxed(&empty_u[U_TM], eph);
                if (lane == 2) mbar_expect_tx(&full_u[U_TM], RG * (rowB + lrowB));
                __syncwarp();
                if (lane == 2) bulk_g2s(tm, in + (size_t)rtm * rowB, RG * rowB, &full_u[U_TM]);
                else if (lane == 3) bulk_g2s(links + (size_t)LK_TM * RG * lrowB, U + (size_t)(6 + 1 - A.par) * ublk + (size_t)rtm * lrowB, RG * lrowB, &full_u[U_TM]);
                mbar_wait_relaxed(&empty_u[U_ZM], eph);
                if (lane == 4) {
                    mbar_expect_tx(&full_u[U_ZM], RG * lrowB);
                    bulk_g2s(links + (size_t)LK_ZM * RG * lrowB, U + (size_t)(4 + 1 - A.par) * ublk + (size_t)rzm * lrowB, RG * lrowB, &full_u[U_ZM]);
                }
                __syncwarp();
                while (issued <= a + 2) {
                    const uint32_t d = issued - a;   // 0, 1, 2 = z-1, z, z+1
                    const uint32_t zz = d == 0 ? wdec(z, A.Lz) : (d == 1 ? z : winc(z, A.Lz));
                    const uint32_t w = issued % 3, use = issued / 3;
                    mbar_wait_relaxed(&empty_w[w], (use & 1) ^ 1);
                    if (lane == 5 + d) {
                        mbar_expect_tx(&full_w[w], RG * rowB);
                        bulk_g2s(planes + (size_t)w * RG * rowB, in + (size_t)(y0 + A.Ly * (zz + A.Lz * t)) * rowB, RG * rowB, &full_w[w]);
                    }
                    __syncwarp();
                    ++issued;
                }
            } else {
                const bool lo = y0 == 0;
                const uint32_t zt = A.Ly * (z + A.Lz * t);
                const uint32_t rm = (lo ? A.Ly - 1 : y0 - 1) + zt, rp = (y0 + RG == A.Ly ? 0 : y0 + RG) + zt;
                mbar_wait_relaxed(&empty_u[U_Y], eph);
                if (lane == 0) mbar_expect_tx(&full_u[U_Y], 2 * rowB + 2 * RG * lrowB);
                __syncwarp();
                char* lym = links + (size_t)LK_YM * RG * lrowB;
                const char* uym = U + (size_t)(2 + 1 - A.par) * ublk;
                if (lane == 0) bulk_g2s(halo, in + (size_t)rm * rowB, rowB, &full_u[U_Y]);
                else if (lane == 1) bulk_g2s(halo + rowB, in + (size_t)rp * rowB, rowB, &full_u[U_Y]);
                else if (lane == 2) bulk_g2s(lym, uym + (size_t)rm * lrowB, (lo ? 1u : RG) * lrowB, &full_u[U_Y]);
                else if (lane == 3 && lo && RG > 1) bulk_g2s(lym + lrowB, uym + (size_t)row0 * lrowB, (RG - 1) * lrowB, &full_u[U_Y]);
                else if (lane == 4) bulk_g2s(links + (size_t)LK_YP * RG * lrowB, U + (size_t)(2 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_Y]);
                mbar_wait_relaxed(&empty_u[U_XZ], eph);
                if (lane == 5) mbar_expect_tx(&full_u[U_XZ], 3 * RG * lrowB);
                __syncwarp();
                if (lane == 5) bulk_g2s(links + (size_t)LK_XM * RG * lrowB, U + (size_t)(0 + 1 - A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_XZ]);
                else if (lane == 6) bulk_g2s(links + (size_t)LK_XP * RG * lrowB, U + (size_t)(0 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_XZ]);
                else if (lane == 7) bulk_g2s(links + (size_t)LK_ZP * RG * lrowB, U + (size_t)(4 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_XZ]);
            }
        }
    } else if (warp >= ncw) {
        // ================= producer warps ================================================================
        // One thread can start a bulk copy only every ~280 ns (measured with a stand-alone streaming probe; the copy engine
        // itself takes 8 issuers in parallel at 85-92 GB/s per SM), and a step needs 13-14 copies, so the units are
        // dealt to FOUR producer warps, each walking the steps on its own and waiting only for its own buffers:
        //   P0: U1 {T+ rows, link t+}, U3 {link z-}      P1: U2 {T- rows, link t-}, window planes
        //   P2: U4 {halo rows, link y-}                  P3: U4 {link y+}, U5 {links x-, x+, z+}
        const uint32_t role = warp - ncw;
        const char* in = reinterpret_cast<const char*>(A.in);
        const char* U = reinterpret_cast<const char*>(A.U);
        const size_t ublk = (size_t)RECON * A.Vh * sizeof(T);   // bytes of one (mu, parity) link array
        uint32_t issued = 0, a = 0, prev = NO_STEP;
        for (uint32_t s = s_first, k = 0; s != NO_STEP; prev = s, s = next_step(s, A.chunk, A.steps), ++k) {
            const uint32_t col = s / A.Lz, z = s - col * A.Lz;
            const uint32_t yb = col % A.gy, t = A.t0 + col / A.gy, y0 = yb * RG;
            if (k > 0) a += continues(prev, s, A.Lz) ? 1u : 3u;
            const uint32_t eph = (k & 1) ^ 1;
            const uint32_t row0 = y0 + A.Ly * (z + A.Lz * t);
            if (role == 0) {
                // ---- U1: T+ rows, link t+ = U_t(x) on the output rows
                const uint32_t rtp = y0 + A.Ly * (z + A.Lz * winc(t, A.Lt));
                mbar_wait_relaxed(&empty_u[U_TP], eph);
                if (lane == 0) mbar_expect_tx(&full_u[U_TP], RG * (rowB + lrowB));
                __syncwarp();
                if (lane == 0) bulk_g2s(tp, in + (size_t)rtp * rowB, RG * rowB, &full_u[U_TP]);
                else if (lane == 1) bulk_g2s(links + (size_t)LK_TP * RG * lrowB, U + (size_t)(6 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_TP]);
                // ---- U3: link z- = U_z(x - z^) on the z-1 rows of the other parity
                const uint32_t rzm = y0 + A.Ly * (wdec(z, A.Lz) + A.Lz * t);
                mbar_wait_relaxed(&empty_u[U_ZM], eph);
                if (lane == 0) {
                    mbar_expect_tx(&full_u[U_ZM], RG * lrowB);
                    bulk_g2s(links + (size_t)LK_ZM * RG * lrowB, U + (size_t)(4 + 1 - A.par) * ublk + (size_t)rzm * lrowB, RG * lrowB, &full_u[U_ZM]);
                }
                __syncwarp();
            } else if (role == 1) {
                // ---- U2: T- rows, link t- = U_t(x - t^) on the t-1 rows of the other parity
                const uint32_t rtm = y0 + A.Ly * (z + A.Lz * wdec(t, A.Lt));
                mbar_wait_relaxed(&empty_u[U_TM], eph);
                if (lane == 0) mbar_expect_tx(&full_u[U_TM], RG * (rowB + lrowB));
                __syncwarp();
                if (lane == 0) bulk_g2s(tm, in + (size_t)rtm * rowB, RG * rowB, &full_u[U_TM]);
                else if (lane == 1) bulk_g2s(links + (size_t)LK_TM * RG * lrowB, U + (size_t)(6 + 1 - A.par) * ublk + (size_t)rtm * lrowB, RG * lrowB, &full_u[U_TM]);
                // ---- window planes up to sequence number a + 2 (one per step; three at a column start)
                while (issued <= a + 2) {
                    const uint32_t d = issued - a;   // 0, 1, 2 = z-1, z, z+1
                    const uint32_t zz = d == 0 ? wdec(z, A.Lz) : (d == 1 ? z : winc(z, A.Lz));
                    const uint32_t w = issued % 3, use = issued / 3;
                    mbar_wait_relaxed(&empty_w[w], (use & 1) ^ 1);
                    if (lane == 0) {
                        mbar_expect_tx(&full_w[w], RG * rowB);
                        bulk_g2s(planes + (size_t)w * RG * rowB, in + (size_t)(y0 + A.Ly * (zz + A.Lz * t)) * rowB, RG * rowB, &full_w[w]);
                    }
                    __syncwarp();
                    ++issued;
                }
            } else if (role == 2) {
                // ---- U4 (with P3): halo rows y0-1, y0+RG of the centre plane; link y- = U_y(x - y^) on rows y0-1 ..
                //      y0+RG-2 of the other parity (one copy unless row y0-1 wraps around)
                const bool lo = y0 == 0;
                const uint32_t zt = A.Ly * (z + A.Lz * t);
                const uint32_t rm = (lo ? A.Ly - 1 : y0 - 1) + zt, rp = (y0 + RG == A.Ly ? 0 : y0 + RG) + zt;
                mbar_wait_relaxed(&empty_u[U_Y], eph);
                if (lane == 0) mbar_expect_tx(&full_u[U_Y], 2 * rowB + 2 * RG * lrowB);   // includes P3's y+ copy
                __syncwarp();
                char* lym = links + (size_t)LK_YM * RG * lrowB;
                const char* uym = U + (size_t)(2 + 1 - A.par) * ublk;
                if (lane == 0) bulk_g2s(halo, in + (size_t)rm * rowB, rowB, &full_u[U_Y]);
                else if (lane == 1) bulk_g2s(halo + rowB, in + (size_t)rp * rowB, rowB, &full_u[U_Y]);
                else if (lane == 2) bulk_g2s(lym, uym + (size_t)rm * lrowB, (lo ? 1u : RG) * lrowB, &full_u[U_Y]);
                else if (lane == 3 && lo && RG > 1) bulk_g2s(lym + lrowB, uym + (size_t)row0 * lrowB, (RG - 1) * lrowB, &full_u[U_Y]);
            } else {
                // ---- link y+ = U_y(x) (part of U4: P2 has announced its bytes), then
                // ---- U5: links x- = U_x(x - x^) (same rows, other parity), x+ = U_x(x), z+ = U_z(x)
                mbar_wait_relaxed(&empty_u[U_Y], eph);
                if (lane == 0) bulk_g2s(links + (size_t)LK_YP * RG * lrowB, U + (size_t)(2 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_Y]);
                mbar_wait_relaxed(&empty_u[U_XZ], eph);
                if (lane == 0) mbar_expect_tx(&full_u[U_XZ], 3 * RG * lrowB);
                __syncwarp();
                if (lane == 0) bulk_g2s(links + (size_t)LK_XM * RG * lrowB, U + (size_t)(0 + 1 - A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_XZ]);
                else if (lane == 1) bulk_g2s(links + (size_t)LK_XP * RG * lrowB, U + (size_t)(0 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_XZ]);
                else if (lane == 2) bulk_g2s(links + (size_t)LK_ZP * RG * lrowB, U + (size_t)(4 + A.par) * ublk + (size_t)row0 * lrowB, RG * lrowB, &full_u[U_XZ]);
            }
        }
    } else if constexpr (ST == 2) {
        // ================= consumers, two sites per thread: thread i = (row j, pair p, column r) =========
        typedef ulonglong2 pv;
        using namespace wdp;
        const uint32_t i = threadIdx.x;
        const bool active = i < nct;
        const uint32_t H = SW, cs = H * nr;                       // pairs per row, elements per complex of a row
        const uint32_t sidx = i / nr, r = i - sidx * nr;
        const uint32_t j = sidx / H, p = sidx - j * H;
        const uint32_t lrowV = lrowB / 16;
        const uint32_t e0 = p * nr + r;
        const pv* const Pl = reinterpret_cast<const pv*>(planes);
        const pv* const Tp = reinterpret_cast<const pv*>(tp) + (size_t)j * rowS;
        const pv* const Tm = reinterpret_cast<const pv*>(tm) + (size_t)j * rowS;
        const pv* const Hl = reinterpret_cast<const pv*>(halo);
        const pv* const Lk = reinterpret_cast<const pv*>(links) + (size_t)j * lrowV;
        const uint32_t lblk = RG * lrowV;
        const uint32_t planeV = RG * rowS;
        if (A.zero_rows) {
            const vec z4 = {};
            for (uint32_t row = blockIdx.x; row < A.zero_rows; row += gridDim.x)
                for (uint32_t v = i; v < rowS; v += ncw * 32) A.out[(size_t)row * rowS + v] = z4;
        }
        const f2 a2 = mk2(A.a, A.a), b2 = mk2(A.b, A.b);
        uint32_t a = 0, prev = NO_STEP;
        for (uint32_t s = s_first, k = 0; s != NO_STEP; prev = s, s = next_step(s, A.chunk, A.steps), ++k) {
            const uint32_t col = s / A.Lz, z = s - col * A.Lz;
            const uint32_t yb = col % A.gy, t = A.t0 + col / A.gy, y0 = yb * RG;
            if (k > 0) a += continues(prev, s, A.Lz) ? 1u : 3u;
            const uint32_t s_next = next_step(s, A.chunk, A.steps);
            const bool switch_next = s_next != NO_STEP && !continues(s, s_next, A.Lz);
            const uint32_t ph = k & 1;
            const size_t own = (size_t)(y0 + A.Ly * (z + A.Lz * t) + j) * rowS;
            cx2 acc[12];
            if (EPI >= EPI_XPAY && active) {
#pragma unroll
                for (uint32_t c = 0; c < 12; ++c) {
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in2 + own + c * cs + e0));
                    if (EPI == EPI_SIGMA) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in3 + own + c * cs + e0));
                }
            }
            const uint32_t wm = a % 3, wc = (a + 1) % 3, wp = (a + 2) % 3;
            const pv* const Pm = Pl + (size_t)wm * planeV + (size_t)j * rowS;
            const pv* const Pc = Pl + (size_t)wc * planeV + (size_t)j * rowS;
            const pv* const Pp = Pl + (size_t)wp * planeV + (size_t)j * rowS;
            // rows with bb = 1 have their +x neighbour one pair up and their -x neighbour in the same pair; bb = 0 the
            // other way round.  A step past the half row lands on the pair at the other end, lanes exchanged.
            const uint32_t bb = (y0 + j + z + t + A.par) & 1;
            const uint32_t pp = bb ? (p + 1 == H ? 0u : p + 1) : p;
            const uint32_t pm = bb ? p : (p == 0 ? H - 1 : p - 1);
            const bool swp_p = bb && p + 1 == H, swp_m = !bb && p == 0;
            const pv* const ym = j == 0 ? Hl : Pc - rowS;
            const pv* const yp = j == RG - 1 ? Hl + rowS : Pc + rowS;
            PairOps oa, ob;
            // direction order t+, t-, z-, y-, y+, x-, x+, z+ (that of every hop kernel); loads one direction ahead
            mbar_wait(&full_u[U_TP], ph);
            if (active) pair_load<RECON>(oa, Tp, cs, e0, Lk + LK_TP * lblk, H, p);
            mbar_wait(&full_u[U_TM], ph);
            if (active) {
                pair_load<RECON>(ob, Tm, cs, e0, Lk + LK_TM * lblk, H, p);
                pair_compute<RECON, 3, true, DAG, true>(oa, acc);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_u[U_TP]);
            mbar_wait(&full_u[U_ZM], ph);
            mbar_wait(&full_w[wm], (a / 3) & 1);
            if (active) {
                pair_load<RECON>(oa, Pm, cs, e0, Lk + LK_ZM * lblk, H, p);
                pair_compute<RECON, 3, false, DAG>(ob, acc);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_u[U_TM]);
            mbar_wait(&full_u[U_Y], ph);
            mbar_wait(&full_w[wc], ((a + 1) / 3) & 1);
            if (active) {
                pair_load<RECON>(ob, ym, cs, e0, Lk + LK_YM * lblk, H, p);
                pair_compute<RECON, 2, false, DAG>(oa, acc);
            }
            __syncwarp();
            if (lane == 0) { mbar_arrive(&empty_u[U_ZM]); mbar_arrive(&empty_w[wm]); }
            if (active) {
                pair_load<RECON>(oa, yp, cs, e0, Lk + LK_YP * lblk, H, p);
                pair_compute<RECON, 1, false, DAG>(ob, acc);
            }
            mbar_wait(&full_u[U_XZ], ph);
            mbar_wait(&full_w[wp], ((a + 2) / 3) & 1);
            if (active) {
                pair_load<RECON>(ob, Pc, cs, pm * nr + r, Lk + LK_XM * lblk, H, pm);
                pair_compute<RECON, 1, true, DAG>(oa, acc);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_u[U_Y]);
            if (active) {
                pair_load<RECON>(oa, Pc, cs, pp * nr + r, Lk + LK_XP * lblk, H, p);
                pair_compute<RECON, 0, false, DAG, false, true>(ob, acc, swp_m);
                pair_load<RECON>(ob, Pp, cs, e0, Lk + LK_ZP * lblk, H, p);
                pair_compute<RECON, 0, true, DAG, false, true>(oa, acc, swp_p);
                pair_compute<RECON, 2, true, DAG>(ob, acc);
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&empty_u[U_XZ]);
                if (switch_next) { mbar_arrive(&empty_w[wc]); mbar_arrive(&empty_w[wp]); }
            }
            // ---- epilogue and store
            if (active) {
                [[maybe_unused]] cx2 qv[12];
                if (EPI >= EPI_XPAY) {
                    ldg_spinor(reinterpret_cast<const pv*>(A.in2) + own, cs, e0, qv);
#pragma unroll
                    for (int q = 0; q < 12; ++q) {
                        acc[q].re = fma2(b2, acc[q].re, mul2(a2, qv[q].re));
                        acc[q].im = fma2(b2, acc[q].im, mul2(a2, qv[q].im));
                    }
                    if (EPI == EPI_OMEGA) {  // <t, s>, <t, t> with t = acc, s = qv
                        f2 s0 = zero2(), s1 = zero2(), s2 = zero2();
#pragma unroll
                        for (int q = 0; q < 12; ++q) {
                            s0 = fma2(acc[q].re, qv[q].re, s0);  s0 = fma2(acc[q].im, qv[q].im, s0);
                            s1 = fma2(acc[q].re, qv[q].im, s1);  s1 = fma2(neg2(acc[q].im), qv[q].re, s1);
                            s2 = fma2(acc[q].re, acc[q].re, s2); s2 = fma2(acc[q].im, acc[q].im, s2);
                        }
                        float lo, hi;
                        un2(s0, lo, hi); dsum[0] += (double)lo + (double)hi;
                        un2(s1, lo, hi); dsum[1] += (double)lo + (double)hi;
                        un2(s2, lo, hi); dsum[2] += (double)lo + (double)hi;
                    }
                }
                if (EPI == EPI_SIGMA) {  // <r~, v> with v = acc
                    ldg_spinor(reinterpret_cast<const pv*>(A.in3) + own, cs, e0, qv);
                    f2 s0 = zero2(), s1 = zero2();
#pragma unroll
                    for (int q = 0; q < 12; ++q) {
                        s0 = fma2(qv[q].re, acc[q].re, s0);  s0 = fma2(qv[q].im, acc[q].im, s0);
                        s1 = fma2(qv[q].re, acc[q].im, s1);  s1 = fma2(neg2(qv[q].im), acc[q].re, s1);
                    }
                    float lo, hi;
                    un2(s0, lo, hi); dsum[0] += (double)lo + (double)hi;
                    un2(s1, lo, hi); dsum[1] += (double)lo + (double)hi;
                }
                st_spinor(reinterpret_cast<pv*>(A.out) + own, cs, e0, acc);
            }
        }
    } else {
        // ================= consumers: thread i = (site s of the step, column r) ==========================
        const uint32_t i = threadIdx.x;
        const bool active = i < nct;
        const uint32_t sidx = i / nr, r = i - sidx * nr;
        const uint32_t j = sidx / Lxh, xh = sidx - j * Lxh;       // row inside the step, site inside the row
        const uint32_t lrowV = lrowB / 16;
        const uint32_t e0 = xh * nr + r;
        const vec* const Pl = reinterpret_cast<const vec*>(planes);
        const vec* const Tp = reinterpret_cast<const vec*>(tp) + (size_t)j * rowS;
        const vec* const Tm = reinterpret_cast<const vec*>(tm) + (size_t)j * rowS;
        const vec* const Hl = reinterpret_cast<const vec*>(halo);
        const vec* const Lk = reinterpret_cast<const vec*>(links) + (size_t)j * lrowV;
        const uint32_t lblk = RG * lrowV;    // 16-byte units of one link block
        const uint32_t planeV = RG * rowS;
        // SF: the stored t = 0 slice of the output stays zero
        if (A.zero_rows) {
            const vec z4 = {};
            for (uint32_t row = blockIdx.x; row < A.zero_rows; row += gridDim.x)
                for (uint32_t v = i; v < rowS; v += ncw * 32) A.out[(size_t)row * rowS + v] = z4;
        }
        uint32_t a = 0, prev = NO_STEP;
        for (uint32_t s = s_first, k = 0; s != NO_STEP; prev = s, s = next_step(s, A.chunk, A.steps), ++k) {
            const uint32_t col = s / A.Lz, z = s - col * A.Lz;
            const uint32_t yb = col % A.gy, t = A.t0 + col / A.gy, y0 = yb * RG;
            if (k > 0) a += continues(prev, s, A.Lz) ? 1u : 3u;
            const uint32_t s_next = next_step(s, A.chunk, A.steps);
            const bool switch_next = s_next != NO_STEP && !continues(s, s_next, A.Lz);
            const uint32_t ph = k & 1;
            const size_t own = (size_t)(y0 + A.Ly * (z + A.Lz * t) + j) * rowS;
            cx<T> acc[12];
            if (EPI >= EPI_XPAY && active) {
#pragma unroll
                for (uint32_t c = 0; c < (ST == 1 ? 3u : NCH); ++c) {
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in2 + own + c * rowV + e0));
                    if (EPI == EPI_SIGMA || EPI == EPI_OMEGA_RHO) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.in3 + own + c * rowV + e0));
                }
            }
            const uint32_t wm = a % 3, wc = (a + 1) % 3, wp = (a + 2) % 3;
            const vec* const Pm = Pl + (size_t)wm * planeV + (size_t)j * rowS;
            const vec* const Pc = Pl + (size_t)wc * planeV + (size_t)j * rowS;
            const vec* const Pp = Pl + (size_t)wp * planeV + (size_t)j * rowS;
            // ---- t+
            mbar_wait(&full_u[U_TP], ph);
            if (active) dir_smem<T, RECON, ST, 3, true, DAG, true>(Tp, rowV, e0, Lk + LK_TP * lblk, Lxh, xh, acc);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_u[U_TP]);
            // ---- t-
            mbar_wait(&full_u[U_TM], ph);
            if (active) dir_smem<T, RECON, ST, 3, false, DAG>(Tm, rowV, e0, Lk + LK_TM * lblk, Lxh, xh, acc);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_u[U_TM]);
            // ---- z-
            mbar_wait(&full_u[U_ZM], ph);
            mbar_wait(&full_w[wm], (a / 3) & 1);
            if (active) dir_smem<T, RECON, ST, 2, false, DAG>(Pm, rowV, e0, Lk + LK_ZM * lblk, Lxh, xh, acc);
            __syncwarp();
            if (lane == 0) { mbar_arrive(&empty_u[U_ZM]); mbar_arrive(&empty_w[wm]); }
            // ---- y-, y+
            mbar_wait(&full_u[U_Y], ph);
            mbar_wait(&full_w[wc], ((a + 1) / 3) & 1);
            if (active) {
                const vec* ym = j == 0 ? Hl : Pc - rowS;
                const vec* yp = j == RG - 1 ? Hl + rowS : Pc + rowS;
                dir_smem<T, RECON, ST, 1, false, DAG>(ym, rowV, e0, Lk + LK_YM * lblk, Lxh, xh, acc);
                dir_smem<T, RECON, ST, 1, true, DAG>(yp, rowV, e0, Lk + LK_YP * lblk, Lxh, xh, acc);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_u[U_Y]);
            // ---- x-, x+, z+
            [[maybe_unused]] cx<T> qv[12];
            if (EPI >= EPI_XPAY && active) { if (ST) wdh::h16_load<true>(A.in2 + own, rowV, e0, qv); else load_spinor(A.in2 + own, rowV, e0, qv); }
            mbar_wait(&full_u[U_XZ], ph);
            mbar_wait(&full_w[wp], ((a + 2) / 3) & 1);
            if (active) {
                const uint32_t bb = (y0 + j + z + t + A.par) & 1;
                const uint32_t xp = bb ? winc(xh, Lxh) : xh;   // xh of the +x neighbour
                const uint32_t xm = bb ? xh : wdec(xh, Lxh);   // xh of the -x neighbour
                dir_smem<T, RECON, ST, 0, false, DAG>(Pc, rowV, xm * nr + r, Lk + LK_XM * lblk, Lxh, xm, acc);
                dir_smem<T, RECON, ST, 0, true, DAG>(Pc, rowV, xp * nr + r, Lk + LK_XP * lblk, Lxh, xh, acc);
                dir_smem<T, RECON, ST, 2, true, DAG>(Pp, rowV, e0, Lk + LK_ZP * lblk, Lxh, xh, acc);
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&empty_u[U_XZ]);
                if (switch_next) { mbar_arrive(&empty_w[wc]); mbar_arrive(&empty_w[wp]); }
            }
            // ---- epilogue and store
            if (active) {
                if (EPI >= EPI_XPAY) {
#pragma unroll
                    for (int q = 0; q < 12; ++q) {
                        acc[q].re = fma(A.b, acc[q].re, A.a * qv[q].re);
                        acc[q].im = fma(A.b, acc[q].im, A.a * qv[q].im);
                    }
                    if (EPI == EPI_OMEGA || EPI == EPI_OMEGA_RHO) {  // <t, s>, <t, t> with t = acc, s = qv
                        T s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
                        for (int q = 0; q < 12; ++q) {
                            s0 = fma(acc[q].re, qv[q].re, s0);  s0 = fma(acc[q].im, qv[q].im, s0);
                            s1 = fma(acc[q].re, qv[q].im, s1);  s1 = fma(-acc[q].im, qv[q].re, s1);
                            s2 = fma(acc[q].re, acc[q].re, s2); s2 = fma(acc[q].im, acc[q].im, s2);
                        }
                        dsum[0] += (double)s0; dsum[1] += (double)s1; dsum[2] += (double)s2;
                    }
                    if constexpr (EPI == EPI_OMEGA_RHO && ST == 0) {  // <rt, s>, <rt, t> with rt = in3, two components at a time
                        T s3 = 0, s4 = 0, s5 = 0, s6 = 0;
#pragma unroll
                        for (int c = 0; c < 6; ++c) {
                            const float4 w = __ldg(A.in3 + own + c * rowV + e0);
                            const cx<T> g0 = {w.x, w.y}, g1 = {w.z, w.w};
                            s3 = fma(g0.re, qv[2 * c].re, s3);  s3 = fma(g0.im, qv[2 * c].im, s3);
                            s4 = fma(g0.re, qv[2 * c].im, s4);  s4 = fma(-g0.im, qv[2 * c].re, s4);
                            s5 = fma(g0.re, acc[2 * c].re, s5); s5 = fma(g0.im, acc[2 * c].im, s5);
                            s6 = fma(g0.re, acc[2 * c].im, s6); s6 = fma(-g0.im, acc[2 * c].re, s6);
                            s3 = fma(g1.re, qv[2 * c + 1].re, s3);  s3 = fma(g1.im, qv[2 * c + 1].im, s3);
                            s4 = fma(g1.re, qv[2 * c + 1].im, s4);  s4 = fma(-g1.im, qv[2 * c + 1].re, s4);
                            s5 = fma(g1.re, acc[2 * c + 1].re, s5); s5 = fma(g1.im, acc[2 * c + 1].im, s5);
                            s6 = fma(g1.re, acc[2 * c + 1].im, s6); s6 = fma(-g1.im, acc[2 * c + 1].re, s6);
                        }
                        dsum[3] += (double)s3; dsum[4] += (double)s4; dsum[5] += (double)s5; dsum[6] += (double)s6;
                    }
                }
                if (EPI == EPI_SIGMA) {  // <r~, v> with v = acc
                    if (ST) wdh::h16_load<true>(A.in3 + own, rowV, e0, qv); else load_spinor(A.in3 + own, rowV, e0, qv);
                    T s0 = 0, s1 = 0;
#pragma unroll
                    for (int q = 0; q < 12; ++q) {
                        s0 = fma(qv[q].re, acc[q].re, s0);  s0 = fma(qv[q].im, acc[q].im, s0);
                        s1 = fma(qv[q].re, acc[q].im, s1);  s1 = fma(-qv[q].im, acc[q].re, s1);
                    }
                    dsum[0] += (double)s0; dsum[1] += (double)s1;
                }
                if (ST) wdh::h16_store(A.out + own, rowV, e0, acc); else store_spinor(A.out + own, rowV, e0, acc);
            }
        }
    }
    if (EPI >= EPI_SIGMA) {
        // per-column sums of this CTA -> one partial per (column, value); the last CTA adds the partials in a fixed
        // order and runs the scalar recurrence (as wd_hop_tma.cu)
        constexpr int K = EPI == EPI_SIGMA ? 2 : (EPI == EPI_OMEGA_RHO ? 7 : 3);
        __syncthreads();  // every bulk copy has been consumed: the staging area is free
        double* red = reinterpret_cast<double*>(base);
        if (threadIdx.x < nct) {
#pragma unroll
            for (int q = 0; q < K; ++q) red[q * nct + threadIdx.x] = dsum[q];
        }
        __syncthreads();
        const uint32_t nwarps = blockDim.x >> 5;
        for (uint32_t item = warp; item < nr * K; item += nwarps) {
            const uint32_t col = item / K, q = item - col * K;
            double v = 0.0;
            for (uint32_t ss = lane; ss < RG * SW; ss += 32) v += red[q * nct + ss * nr + col];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) A.rb.partials[(size_t)item * gridDim.x + blockIdx.x] = v;
        }
        double* tot = red + K * nct;
        volatile uint32_t* is_last = reinterpret_cast<volatile uint32_t*>(tot + nr * K);
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) *is_last = (atomicAdd(A.rb.ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
        __syncthreads();
        if (*is_last == 0u) return;
        __threadfence();
        for (uint32_t item = warp; item < nr * K; item += nwarps) {
            const double* p = A.rb.partials + (size_t)item * gridDim.x;
            double v = 0.0;
            for (uint32_t g = lane; g < gridDim.x; g += 32) v += __ldcg(p + g);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) tot[item] = v;
        }
        __syncthreads();
        if (threadIdx.x < nr)
            wdblas::finalize_column<EPI == EPI_SIGMA ? wdblas::K_SIGMA : (EPI == EPI_OMEGA_RHO ? wdblas::K_OMEGA_RHO : wdblas::K_OMEGA)>(A.rb.scal, (int)threadIdx.x, tot + threadIdx.x * K);
        if (threadIdx.x == 0) *A.rb.ticket = 0u;
    }
}

// ---- host side ----------------------------------------------------------------------------------------------
constexpr size_t kSmemMax = 227 * 1024;

struct Shape {
    uint32_t RG, S, threads;
    size_t smem;
};

// largest row group (a divisor of Ly) whose CTA fits the thread budget and whose buffers fit shared memory
template <typename T, int RECON, int ST>
bool pick_shape(const wd_ctx* c, int n, int max_threads, Shape* sh) {
    const uint32_t Lxh = c->L[0] / 2, Ly = c->L[1];
    const uint32_t cap = c->opt[WD_OPT_HOP_ROWS] > 0 ? (uint32_t)c->opt[WD_OPT_HOP_ROWS] : Ly;
    for (uint32_t RG = Ly; RG >= 1; --RG) {
        if (Ly % RG || RG > cap) continue;
        const uint32_t S = RG * Lxh;
        const uint32_t cthreads = (((ST == 2 ? S / 2 : S) * n + 31) / 32) * 32;   // ST = 2: one thread per site pair
        const uint32_t pthreads = ST == 2 ? 64 : 128;   // producer warps: two in the P32 form, else four
        if ((int)(cthreads + pthreads) > max_threads) continue;
        const size_t rowB = ST == 1 ? (size_t)wdh::h16_row_vecs(Lxh * n) * 16 : (size_t)Lxh * n * 16 * Vec<T>::NCH;
        const size_t lrowB = (size_t)Lxh * RECON * sizeof(T);
        const size_t smem = 128 + (5 * (size_t)RG + 2) * rowB + 8 * (size_t)RG * lrowB;
        if (smem > kSmemMax) continue;
        // the epilogue's reduction scratch (3 sums per consumer thread + totals) reuses the staging area
        if ((size_t)(7 * S * n + 7 * WD_MAX_RHS + 2) * sizeof(double) > smem - 128) continue;
        sh->RG = RG; sh->S = S; sh->threads = cthreads + pthreads; sh->smem = smem;
        return true;
    }
    return false;
}

template <typename T, int RECON, bool DAG, int EPI, int MAXT, int LXH, int NR, int RGT, int ST>
int launch_one(wd_ctx* c, const ZmArgs<T>& A, const Shape& sh, unsigned G) {
    auto kern = hop_zm_kernel<T, RECON, DAG, EPI, MAXT, LXH, NR, RGT, ST>;
    WD_CUDA_CHECK(c, wd_ensure_smem_attr(c, (const void*)kern, (int)kSmemMax));
    kern<<<G, sh.threads, sh.smem, c->stream>>>(A);
    return WD_OK;
}

template <typename T, int RECON, int MAXT, int LXH, int NR, int RGT, int ST>
int launch_epi(wd_ctx* c, const ZmArgs<T>& A, const Shape& sh, unsigned G, int dag, int epi) {
#define WD_ZM_CASE(D, E) return launch_one<T, RECON, D, E, MAXT, LXH, NR, RGT, ST>(c, A, sh, G)
    if (epi == EPI_OMEGA_RHO) {
        if constexpr (ST == 0) {
            if (dag) WD_ZM_CASE(true, EPI_OMEGA_RHO);
            else WD_ZM_CASE(false, EPI_OMEGA_RHO);
        }
        return 1;
    }
    if (dag) {
        if (epi == EPI_NONE) WD_ZM_CASE(true, EPI_NONE);
        else if (epi == EPI_XPAY) WD_ZM_CASE(true, EPI_XPAY);
        else if (epi == EPI_SIGMA) WD_ZM_CASE(true, EPI_SIGMA);
        else WD_ZM_CASE(true, EPI_OMEGA);
    } else {
        if (epi == EPI_NONE) WD_ZM_CASE(false, EPI_NONE);
        else if (epi == EPI_XPAY) WD_ZM_CASE(false, EPI_XPAY);
        else if (epi == EPI_SIGMA) WD_ZM_CASE(false, EPI_SIGMA);
        else WD_ZM_CASE(false, EPI_OMEGA);
    }
#undef WD_ZM_CASE
}

template <typename T, int RECON, int MAXT, int ST>
int launch_zm(wd_ctx* c, int dag, int n, int par, const wd_hop_ops& o, const T* U) {
    Shape sh;
    if (ST == 1 && ((c->L[0] / 2) * n) % 4 != 0) return 1;   // the H16 scale chunk must keep rows 16-byte aligned
    if (!pick_shape<T, RECON, ST>(c, n, MAXT, &sh)) return 1;
    ZmArgs<T> A;
    A.in = (const typename Vec<T>::type*)o.in;
    A.out = (typename Vec<T>::type*)o.out;
    A.in2 = (const typename Vec<T>::type*)o.in2;
    A.in3 = (const typename Vec<T>::type*)o.in3;
    A.U = U;
    A.rb = wdblas::RedBuf{c->d_scal, c->d_partials, c->d_ticket};
    A.done = o.check_done ? c->d_scal + wdblas::G_DONE : nullptr;
    A.Lxh = c->L[0] / 2; A.Ly = c->L[1]; A.Lz = c->L[2]; A.Lt = c->L[3];
    A.Vh = (uint32_t)c->Vh; A.n = (uint32_t)n; A.par = (uint32_t)par;
    A.RG = sh.RG; A.S = sh.S;
    A.gy = A.Ly / sh.RG;
    A.t0 = c->bc == WD_BC_SF ? 1u : 0u;
    A.steps = A.gy * (A.Lt - A.t0) * A.Lz;
    A.zero_rows = c->bc == WD_BC_SF ? A.Ly * A.Lz : 0u;
    A.a = (T)o.a; A.b = (T)o.b;
    // Chunk length: a divisor of gy * Lz, the step distance between the columns of t and t + 1, so that the CTAs
    // working on t-neighbouring columns are at the same z at the same time and the T+- rows one of them copies are
    // still in L2 when the other copies them as its centre plane (with chunks of steps/G = 14.9 steps the two were
    // 6.5 steps = 150 MB of traffic apart at 24^4: ncu r02a, DRAM reads 271 MB against 168 MB algorithmic).  Among
    // those: the smallest makespan, counting 1.5 steps for every window restart.
    {
        const uint32_t period = A.gy * A.Lz, G0 = (uint32_t)c->n_sm;
        double best = 1e30;
        A.chunk = 1;
        for (uint32_t L = 1; L <= period; ++L) {
            if (period % L) continue;
            const uint32_t nch = (A.steps + L - 1) / L, waves = (nch + G0 - 1) / G0;
            const double cost = waves * (L + 1.5 * (1 + (L - 1) / A.Lz));
            if (cost < best) { best = cost; A.chunk = L; }
        }
    }
    const uint32_t nch = (A.steps + A.chunk - 1) / A.chunk;
    const unsigned G = nch < (uint32_t)c->n_sm ? nch : (unsigned)c->n_sm;
    // shapes with a compile-time geometry (the paper-shaped lattices of BASELINE.json at their n_rhs); any other
    // shape runs the same kernel with run-time strides
#define WD_ZM_GEOM(LXH, NR, RGT) if (A.Lxh == LXH && A.n == NR && A.RG == RGT) return launch_epi<T, RECON, MAXT, LXH, NR, RGT, ST>(c, A, sh, G, dag, o.epi)
    WD_ZM_GEOM(12, 5, 6);
    if constexpr (ST == 0) {   // the other shapes of BASELINE.json's sweeps that this kernel serves: 24^4 at n_rhs = 8, 16^4 at n_rhs = 5
        WD_ZM_GEOM(12, 8, 4);
        WD_ZM_GEOM(8, 5, 8);
    }
#undef WD_ZM_GEOM
    return launch_epi<T, RECON, MAXT, 0, 0, 0, ST>(c, A, sh, G, dag, o.epi);
}

}  // namespace

bool wd_hop_zm_serves(const wd_ctx* c, int recon, int n, int storage) {
    if (c->order != WD_ORDER_LINEAR || c->RB != (uint32_t)(c->L[0] / 2)) return false;
    Shape sh;
    if (storage == 2) {
        if (!c->paired_ok) return false;
        return recon == WD_LINK18 ? pick_shape<float, 18, 2>(c, n, 256, &sh) : pick_shape<float, 12, 2>(c, n, 256, &sh);
    }
    if (storage == 1) {
        if (((c->L[0] / 2) * n) % 4 != 0) return false;
        return recon == WD_LINK18 ? pick_shape<float, 18, 1>(c, n, 512, &sh) : pick_shape<float, 12, 1>(c, n, 512, &sh);
    }
    return recon == WD_LINK18 ? pick_shape<float, 18, 0>(c, n, 512, &sh) : pick_shape<float, 12, 0>(c, n, 512, &sh);
}

// The dispatch rule of WD_OPT_HOP_IMPL = 2 for plain fp32 operands: the z-march kernel unless its step is small AND its
// rows are long -- few consumer threads hide little latency, and long rows are what the row-group ring kernel copies well.
// Measured at 24^4, fp32, 18-real links (us per launch, z-march / ring): n = 3: 46.8 / 55.6, 4: 57.9 / 56.2, 5: 59 / 71,
// 6: 83.1 / 73.5, 8: 84.7 / 105.8, 10: 111.7 / 127.6, 12: 160.0 / 135.5, 16: 233.9 / 177.6; at 16^4 the z-march kernel is
// ahead for every n up to 12.
bool wd_hop_zm_preferred(const wd_ctx* c, int recon, int n) {
    if (!wd_hop_zm_serves(c, recon, n, 0)) return false;
    Shape sh;
    if (recon == WD_LINK18) pick_shape<float, 18, 0>(c, n, 512, &sh); else pick_shape<float, 12, 0>(c, n, 512, &sh);
    const size_t rowB = (size_t)(c->L[0] / 2) * n * 96;
    return !(sh.threads - 128 < 320 && rowB >= 6000);
}

// Returns WD_OK if launched, a positive value if this lattice / option set is not served by this kernel (tiled site
// order, fp64, nothing fits): the caller then tries wd_hop_tma.cu's kernel and then the register kernel.
int wd_hop_zm_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o) {
    if (c->order != WD_ORDER_LINEAR || c->RB != (uint32_t)(c->L[0] / 2)) return 1;  // needs the row-major layout
    if (prec != WD_F32) return 1;
    if (o.storage == 1) {
        if (recon == WD_LINK18) return launch_zm<float, 18, 512, 1>(c, dag, n, par, o, c->d_U32[0]);
        return launch_zm<float, 12, 512, 1>(c, dag, n, par, o, c->d_U32[1]);
    }
    if (o.storage == 2) {   // P32: two sites per thread (wd_f2.cuh); 256 threads leave the consumers 255 registers
        if (!c->paired_ok) return 1;
        if (recon == WD_LINK18) return launch_zm<float, 18, 256, 2>(c, dag, n, par, o, c->d_U32P[0]);
        return launch_zm<float, 12, 256, 2>(c, dag, n, par, o, c->d_U32P[1]);
    }
    if (recon == WD_LINK18) return launch_zm<float, 18, 512, 0>(c, dag, n, par, o, c->d_U32[0]);
    return launch_zm<float, 12, 512, 0>(c, dag, n, par, o, c->d_U32[1]);
}
