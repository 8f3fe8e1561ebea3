// wd_internal.h -- context, workspace map and launch helpers shared by the library's .cu files.
// Not part of the public ABI (include/wd.h is).  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>

#include "../../include/wd.h"

#define WD_NDIR 8  // x+, x-, y+, y-, z+, z-, t+, t-

// Bit 31 of nbr[.][0] marks a site that is not dynamical (SF: the stored t=0 slice).
#define WD_SITE_FROZEN 0x80000000u

// A block of inner-solver iterations captured once as a CUDA graph and replayed (wd_solve.cu).
struct wd_graph_entry {
    unsigned long long key;
    cudaGraphExec_t exec;   // null: the block has run once in stream order (function attributes are set), not yet captured
    long long launches;     // kernel launches one replay stands for
    // wd_profile on: the event pairs recorded as nodes of this graph (begin, end, class); every replay re-records them
    // and the solver adds their times up before the next replay
    std::vector<cudaEvent_t> ev;
    std::vector<int> cls;
};

struct wd_ctx {
    int L[4];
    long V, Vh;
    double kappa;
    int bc;
    int max_rhs;
    cudaStream_t stream;
    int n_sm;

    int order;
    int tile[4];
    // Native layout: sites of a parity are cut into blocks of RB consecutive sites and every block holds its
    // chunks one after the other (spinor: [block][chunk][site in block][rhs] 128-bit elements; links alike).
    // Linear site order with Lx/2 even and max_rhs >= 3: RB = Lx/2, a block is one lattice row (what the staged hop kernel copies
    // in bulk); otherwise RB = V/2, one block, i.e. plain chunk-major.  A site index is stored PACKED in the
    // neighbour table as (block << rb_lg) | offset, 2^rb_lg >= RB, so kernels decode it with a shift and a mask.
    uint32_t RB, rb_lg;

    // host copies of the site tables (uploaded by wd_set_workspace)
    std::vector<int32_t> h_site_of;  // [2][Vh]   canonical site index of (parity, h)
    std::vector<int32_t> h_nbr;      // [2][Vh][8] index (in parity 1-p) of the 8 neighbours of (p, h)

    // workspace
    char* ws;
    size_t ws_bytes;
    bool have_ws, have_gauge;

    // device pointers carved from the workspace
    int32_t* d_site_of;
    int32_t* d_nbr;
    double* d_U64[2];  // [recon] native fp64 links  [mu][parity][R][Vh]
    float* d_U32[2];   // [recon] native fp32 links
    // P32, the x-paired fp32 form (wd_f2.cuh): available in the row-major layout (RB = Lx/2, which is even there)
    bool paired_ok;
    float* d_U32P[2];  // [recon] P32 links (null unless paired_ok)
    // solver scratch
    double* d_scal;        // per-RHS scalars (see wd_solve.cu)
    double* d_partials;    // block partial sums
    size_t partial_doubles; // capacity of d_partials
    double* d_totals;      // 3 * WD_MAX_RHS item totals of the two-kernel reductions
    unsigned int* d_ticket;
    double* h_pinned;      // pinned host mirror for convergence polling (cudaMallocHost, small)
    char* d_solver;        // remaining scratch for solver vectors and host-path staging
    size_t solver_bytes;

    double* d_hist;        // caller's residual-history buffer (wd_set_residual_history), null = off
    int hist_cap;          // its capacity in rows of WD_MAX_RHS doubles

    int opt[WD_OPT_N];  // tunables (wd_set_option)

    // CUDA graphs of the inner solver's iteration blocks; dropped whenever an option or the workspace changes
    std::vector<wd_graph_entry> graphs;
    cudaStream_t cap_stream;   // the library's own stream to capture on (the caller's may be the legacy default stream)

    long long launches;
    std::string err;
    // kernels whose MaxDynamicSharedMemorySize attribute has been raised on THIS context's device (function
    // attributes are per device, and a context is bound to one device)
    std::vector<const void*> smem_attr_done;

    // optional per-class device timing (wd_profile): CUDA event pairs around the classed launches
    bool prof_on;
    int prof_depth;                     // open wd_prof_scope brackets: only the outermost records events
    std::vector<cudaEvent_t> prof_ev;   // pairs (begin, end)
    wd_graph_entry* prof_graph;         // set while a graph is being captured: brackets record into its own event list
    double prof_acc_ms[8];              // time per class accumulated from graph replays since the last wd_profile_read
    long long prof_acc_cnt[8];
    std::vector<int> prof_cls;          // class of pair i
    size_t prof_used;                   // pairs used since the last wd_profile_read
};

// RAII bracket: records an event pair on the context's stream around the launches in its scope.
struct wd_prof_scope {
    wd_ctx* c;
    long idx;
    cudaEvent_t g_end;
    wd_prof_scope(wd_ctx* ctx, int cls) : c(ctx), idx(-1), g_end(nullptr) {
        if (c->prof_depth++ > 0 || !c->prof_on) return;
        if (c->prof_graph) {   // capturing: the records become event-record nodes of the graph, readable from outside
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
            c->prof_graph->ev.push_back(a);
            c->prof_graph->ev.push_back(b);
            c->prof_graph->cls.push_back(cls);
            cudaEventRecordWithFlags(a, c->stream, cudaEventRecordExternal);
            g_end = b;
            return;
        }
        if (c->prof_used == c->prof_cls.size()) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
            c->prof_ev.push_back(a);
            c->prof_ev.push_back(b);
            c->prof_cls.push_back(cls);
        }
        idx = (long)c->prof_used++;
        c->prof_cls[idx] = cls;
        cudaEventRecord(c->prof_ev[2 * idx], c->stream);
    }
    ~wd_prof_scope() {
        --c->prof_depth;
        if (g_end) cudaEventRecordWithFlags(g_end, c->stream, cudaEventRecordExternal);
        if (idx >= 0) cudaEventRecord(c->prof_ev[2 * idx + 1], c->stream);
    }
};

static inline uint32_t wd_pack_site(const wd_ctx* c, long h) {
    return (uint32_t)(((h / c->RB) << c->rb_lg) | (h % c->RB));
}

static inline size_t wd_align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// size in bytes of a native HALF-lattice block
static inline size_t wd_half_bytes(const wd_ctx* c, int prec, int n) {
    return (size_t)c->Vh * 24 * (prec == WD_F64 ? 8 : 4) * (size_t)n;   // WD_F32 and WD_F32P: 4 bytes per real
}
static inline bool wd_is_prec(int prec) { return prec == WD_F64 || prec == WD_F32 || prec == WD_F32P; }

static inline int wd_fail(wd_ctx* c, int code, const char* msg) {
    if (c) c->err = msg;
    return code;
}

#define WD_CUDA_CHECK(ctx, expr)                                                     \
    do {                                                                             \
        cudaError_t e__ = (expr);                                                    \
        if (e__ != cudaSuccess) {                                                    \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e__);        \
            return WD_ECUDA;                                                         \
        }                                                                            \
    } while (0)

#define WD_LAUNCH_CHECK(ctx)                                                         \
    do {                                                                             \
        (ctx)->launches++;                                                           \
        cudaError_t e__ = cudaGetLastError();                                        \
        if (e__ != cudaSuccess) {                                                    \
            (ctx)->err = std::string("kernel launch: ") + cudaGetErrorString(e__);   \
            return WD_ECUDA;                                                         \
        }                                                                            \
    } while (0)

// Raise a kernel's dynamic shared-memory limit once per context (i.e. per device).
static inline cudaError_t wd_ensure_smem_attr(wd_ctx* c, const void* kern, int bytes) {
    for (const void* k : c->smem_attr_done)
        if (k == kern) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) c->smem_attr_done.push_back(kern);
    return e;
}

// ---- internal entry points (device pointers, no argument checks) -------------------------------
// wd_hop.cu
// out[h][r] = (xpay ? a * in2 + b * (H in) : H in) on output parity `par`; in/out/in2 half-lattice blocks.
// If dots != nullptr (fp32/fp64), see wd_hop.cu for the fused reductions.
// general form: epi = 0 none, 1 xpay (in2), 2 xpay + sigma = <in3, out> -> alpha, 3 xpay + <out,in2>, <out,out> -> omega
// (2, 3: fp32 only, scalars land in the solver's table);  check_done: no-op when the solver's done flag is set.
struct wd_hop_ops {
    const void* in;
    void* out;
    const void* in2;
    const void* in3;
    double a, b;
    int epi;
    bool check_done;
    int rev;  // 1: sweep the sites from the top (L2 reuse between consecutive kernels)
    int storage = 0;  // 1: spinor blocks in the 16-bit H16 format (wd_h16.cuh); 2: P32 (wd_f2.cuh); z-march kernel only
};
int wd_hop_launch_ex(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o);
// wd_hop_tma.cu: the shared-memory-staged (bulk copy + mbarrier) form; > 0 = not applicable, use the plain kernel
int wd_hop_tma_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o);
bool wd_hop_tma_serves(const wd_ctx* c, int prec, int recon, int n);
// wd_hop.cu: which kernel wd_hop_launch_ex picks for plain operands (WD_HOP_KERNEL_*), without launching anything
int wd_hop_kernel_for(const wd_ctx* c, int prec, int recon, int n);
// wd_solve.cu: the forms the fp32 inner solver takes for (recon, n) under the current options
void wd_inner_forms(const wd_ctx* c, int recon, int n, bool* paired, bool* merged);
// wd_hop_zm.cu: the z-marching sliding-window form (fp32); > 0 = not applicable
int wd_hop_zm_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const wd_hop_ops& o);
// does the z-march kernel serve this (n_rhs, link form, storage) on this context's lattice?
bool wd_hop_zm_serves(const wd_ctx* c, int recon, int n, int storage);
// ... and is it the faster of the two staged kernels there (plain fp32 operands)?
bool wd_hop_zm_preferred(const wd_ctx* c, int recon, int n);
int wd_hop_launch(wd_ctx* c, int prec, int recon, int dag, int n, int par, const void* in, void* out,
                  const void* in2, double a, double b);

// wd_ctx.cu
void wd_graphs_clear(wd_ctx* c);

// wd_layout.cu
int wd_layout_gauge(wd_ctx* c, const double* U);
int wd_layout_pack(wd_ctx* c, int prec, int n, const double* canon, void* native);
int wd_layout_unpack(wd_ctx* c, int prec, int n, const void* native, double* canon);

// wd_solve.cu
size_t wd_solver_scratch_bytes(const wd_ctx* c);
int wd_solve_impl(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_outer,
                  int max_inner, double inner_tol, int recon, wd_solve_info* info);
int wd_solve_dc(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_outer,
                int max_inner, double inner_tol, int recon, wd_solve_info* info);
int wd_inner_solve_f32(wd_ctx* c, int dag, int n, int recon, int max_inner, const double2* R64, double2* Xacc);
// wd_solve_gl.cu
int wd_solve_gl(wd_ctx* c, int flex, int dag, int n, const double* Phi, double* X, double tol, int max_outer, int max_inner,
                double inner_tol, int recon, wd_solve_info* info);
// returns WD_BL_BREAKDOWN (> 0, never seen by the caller of the C ABI) when the block recurrence lost rank: X is then
// the last good iterate of the even sites only and wd_solve_impl runs the default route instead
#define WD_BL_BREAKDOWN 1
int wd_solve_bl(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_iters, wd_solve_info* info);
// wd_solve_h16.cu
bool wd_solve_h16_applies(const wd_ctx* c, int recon, int n);
int wd_solve_h16(wd_ctx* c, int dag, int n, const double* Phi, double* X, double tol, int max_updates, int max_iters,
                 double delta, int recon, wd_solve_info* info);

// wd_force.cu
int wd_force_impl(wd_ctx* c, int n, const double* X, const double* Y, double* F);

// wd_md.cu
int wd_action_impl(wd_ctx* c, int n, int parity_sel, const double* X, double* S_host);
int wd_project_parity_impl(wd_ctx* c, int prec, int n, int parity, void* native);
int wd_refresh_impl(wd_ctx* c, int variant, int n, const double* eta, double* phi);
int wd_md_force_impl(wd_ctx* c, int variant, int n, const double* Phi, double* X, double* Y, double* F, double* S_host,
                     double* tmp, double tol, int max_outer, int max_inner, double inner_tol, int recon,
                     wd_solve_info* info2);
