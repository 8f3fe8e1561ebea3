// wd_ctx.cu -- context life cycle, site tables, workspace map and the argument-checking front of
// every C-ABI entry point declared in include/wd.h.
#include <chrono>
#include <cmath>
#include <cstring>
#include <new>

#include "wd_internal.h"

namespace {

inline long canon_site(const wd_ctx* c, const int x[4]) {
    return x[0] + (long)c->L[0] * (x[1] + (long)c->L[1] * (x[2] + (long)c->L[2] * x[3]));
}

// position of a site inside its parity for the chosen order
long order_index(const wd_ctx* c, const int x[4]) {
    if (c->order == WD_ORDER_LINEAR) return canon_site(c, x) >> 1;
    const int* b = c->tile;
    int nt[4], tc[4], ic[4];
    for (int d = 0; d < 4; ++d) { nt[d] = c->L[d] / b[d]; tc[d] = x[d] / b[d]; ic[d] = x[d] % b[d]; }
    long tile_idx = tc[0] + (long)nt[0] * (tc[1] + (long)nt[1] * (tc[2] + (long)nt[2] * tc[3]));
    long in_tile = ic[0] + (long)b[0] * (ic[1] + (long)b[1] * (ic[2] + (long)b[2] * ic[3]));
    long tile_half = (long)b[0] * b[1] * b[2] * b[3] / 2;
    return tile_idx * tile_half + (in_tile >> 1);
}

void build_tables(wd_ctx* c) {
    const long V = c->V, Vh = c->Vh;
    // row-major blocks need Lx/2 even: a row of 18-real fp32 links is Lx/2 * 72 bytes and must stay 16-byte aligned
    // and only pay when the staged kernel can run at all (n_rhs >= 3): the register kernel is ~8 % faster chunk-major
    c->RB = (c->order == WD_ORDER_LINEAR && (c->L[0] / 2) % 2 == 0 && c->max_rhs >= 3) ? (uint32_t)(c->L[0] / 2) : (uint32_t)Vh;
    c->rb_lg = 0;
    while ((1u << c->rb_lg) < c->RB) ++c->rb_lg;
    c->paired_ok = c->RB == (uint32_t)(c->L[0] / 2) && c->RB % 2 == 0;
    c->h_site_of.assign(2 * Vh, -1);
    c->h_nbr.assign(2 * Vh * WD_NDIR, 0);
    std::vector<int32_t> idx_of(V);
    int x[4];
    for (x[3] = 0; x[3] < c->L[3]; ++x[3])
        for (x[2] = 0; x[2] < c->L[2]; ++x[2])
            for (x[1] = 0; x[1] < c->L[1]; ++x[1])
                for (x[0] = 0; x[0] < c->L[0]; ++x[0]) {
                    const int p = (x[0] + x[1] + x[2] + x[3]) & 1;
                    const long h = order_index(c, x);
                    const long s = canon_site(c, x);
                    c->h_site_of[p * Vh + h] = (int32_t)s;
                    idx_of[s] = (int32_t)h;
                }
    for (x[3] = 0; x[3] < c->L[3]; ++x[3])
        for (x[2] = 0; x[2] < c->L[2]; ++x[2])
            for (x[1] = 0; x[1] < c->L[1]; ++x[1])
                for (x[0] = 0; x[0] < c->L[0]; ++x[0]) {
                    const int p = (x[0] + x[1] + x[2] + x[3]) & 1;
                    const long h = idx_of[canon_site(c, x)];
                    int32_t* nb = &c->h_nbr[(p * Vh + h) * WD_NDIR];
                    for (int mu = 0; mu < 4; ++mu)
                        for (int s = 0; s < 2; ++s) {
                            int y[4] = {x[0], x[1], x[2], x[3]};
                            y[mu] = (y[mu] + (s == 0 ? 1 : c->L[mu] - 1)) % c->L[mu];
                            nb[2 * mu + s] = (int32_t)wd_pack_site(c, idx_of[canon_site(c, y)]);
                        }
                    // SF: the stored t=0 slice is not dynamical.  Its neighbours at t=1 / t=T-1 read it
                    // as the zero field, which is exactly psi(t=0) = psi(t=T) = 0 (reading R6).
                    if (c->bc == WD_BC_SF && x[3] == 0) nb[0] = (int32_t)((uint32_t)nb[0] | WD_SITE_FROZEN);
                }
}

struct WsMap {
    size_t site_of, nbr, u64[2], u32[2], u32p[2], scal, partials, ticket, solver, total;
};

const int kReals[2] = {18, 12};
const size_t kScalDoubles = 64 * WD_MAX_RHS;
// Reducing kernels write n * K partial sums per block, K <= 3, n <= WD_MAX_RHS.  Largest grids: BLAS1 4 x SMs;
// staged hops one CTA per SM; the register hop with fused inner products always runs 32 sites per CTA
// (wd_hop.cu launch_t), i.e. ceil(V/2 / 32) blocks, and checks its grid against this capacity.
size_t partial_doubles(const wd_ctx* c) {
    const size_t blocks = (size_t)c->Vh / 32 + 1 > 4096 ? (size_t)c->Vh / 32 + 1 : 4096;
    return 3 * blocks * WD_MAX_RHS;
}

WsMap ws_map(const wd_ctx* c) {
    WsMap m;
    size_t o = 0;
    m.site_of = o; o += wd_align_up(sizeof(int32_t) * 2 * c->Vh);
    m.nbr = o;     o += wd_align_up(sizeof(int32_t) * 2 * c->Vh * WD_NDIR);
    for (int r = 0; r < 2; ++r) { m.u64[r] = o; o += wd_align_up(sizeof(double) * 4 * c->V * kReals[r]); }
    for (int r = 0; r < 2; ++r) { m.u32[r] = o; o += wd_align_up(sizeof(float) * 4 * c->V * kReals[r]); }
    for (int r = 0; r < 2; ++r) { m.u32p[r] = o; if (c->paired_ok) o += wd_align_up(sizeof(float) * 4 * c->V * kReals[r]); }
    m.scal = o;     o += wd_align_up(sizeof(double) * kScalDoubles);
    m.partials = o; o += wd_align_up(sizeof(double) * partial_doubles(c));
    m.ticket = o;   o += wd_align_up(256);
    m.solver = o;   o += wd_align_up(wd_solver_scratch_bytes(c));
    m.total = o;
    return m;
}

bool bad_n(const wd_ctx* c, int n) { return n < 1 || n > c->max_rhs; }

}  // namespace

void wd_graphs_clear(wd_ctx* c) {
    for (wd_graph_entry& g : c->graphs) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        for (cudaEvent_t e : g.ev) cudaEventDestroy(e);
    }
    c->graphs.clear();
}

extern "C" {

// A library built with extra -D switches (build.py WD_NVCC_DEFINES: the ablation switches of wd_hop_zm.cu) says so here,
// because such a build computes wrong results on purpose.
#ifdef WD_BUILD_DEFINES
const char* wd_version(void) { return "wd 0.1 (sm_100a) MEASUREMENT BUILD: " WD_BUILD_DEFINES; }
#else
const char* wd_version(void) { return "wd 0.1 (sm_100a)"; }
#endif

const char* wd_strerror(int code) {
    switch (code) {
        case WD_OK: return "ok";
        case WD_EINVAL: return "invalid argument";
        case WD_ENOMEM: return "out of memory";
        case WD_ECUDA: return "CUDA error";
        case WD_ENOCONV: return "solver did not reach the tolerance";
        case WD_ESTATE: return "call out of order (workspace or gauge field not set)";
        default: return "unknown error code";
    }
}

const char* wd_last_error(const wd_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

long long wd_launch_count(const wd_ctx* ctx) { return ctx ? ctx->launches : 0; }

int wd_create(wd_ctx** out, const int dims[4], double kappa, int time_bc, int max_rhs, void* cuda_stream) {
    if (!out || !dims) return WD_EINVAL;
    *out = nullptr;
    if (!std::isfinite(kappa)) return WD_EINVAL;
    if (time_bc != WD_BC_PERIODIC && time_bc != WD_BC_SF) return WD_EINVAL;
    if (max_rhs < 1 || max_rhs > WD_MAX_RHS) return WD_EINVAL;
    long V = 1;
    for (int d = 0; d < 4; ++d) {
        if (dims[d] < 2 || (dims[d] & 1)) return WD_EINVAL;
        V *= dims[d];
        if (V > (1L << 30)) return WD_EINVAL;
    }
    if (time_bc == WD_BC_SF && dims[3] < 4) return WD_EINVAL;
    if (6 * V * max_rhs >= (1L << 31)) return WD_EINVAL;  // kernels index 128-bit elements with 32 bits
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return WD_ECUDA;
    }
    wd_ctx* c = new (std::nothrow) wd_ctx();
    if (!c) return WD_ENOMEM;
    for (int d = 0; d < 4; ++d) c->L[d] = dims[d];
    c->V = V;
    c->Vh = V / 2;
    c->kappa = kappa;
    c->bc = time_bc;
    c->max_rhs = max_rhs;
    c->stream = (cudaStream_t)cuda_stream;
    c->n_sm = prop.multiProcessorCount;
    c->order = WD_ORDER_LINEAR;
    for (int d = 0; d < 4; ++d) c->tile[d] = dims[d];
    c->ws = nullptr;
    c->ws_bytes = 0;
    c->have_ws = c->have_gauge = false;
    c->launches = 0;
    c->d_hist = nullptr;
    c->hist_cap = 0;
    for (int k = 0; k < WD_OPT_N; ++k) c->opt[k] = 0;
    // hop CTA shape and register budget: 0 = chosen per launch from n_rhs (wd_hop.cu)
    c->opt[WD_OPT_POLL_EVERY] = 4;
    c->opt[WD_OPT_HOP_IMPL] = 2;
    c->opt[WD_OPT_ALTERNATE_SWEEP] = 1;
    c->opt[WD_OPT_PAIRED] = 0;
    c->opt[WD_OPT_GRAPH] = 1;
    c->opt[WD_OPT_MERGE] = 1;
    c->cap_stream = nullptr;
    c->prof_on = false;
    c->prof_depth = 0;
    c->prof_graph = nullptr;
    for (int k = 0; k < 8; ++k) { c->prof_acc_ms[k] = 0.0; c->prof_acc_cnt[k] = 0; }
    c->prof_used = 0;
    c->h_pinned = nullptr;
    if (cudaMallocHost((void**)&c->h_pinned, sizeof(double) * kScalDoubles) != cudaSuccess) {
        cudaGetLastError();
        delete c;
        return WD_ENOMEM;
    }
    try {
        build_tables(c);
    } catch (const std::bad_alloc&) {
        cudaFreeHost(c->h_pinned);
        delete c;
        return WD_ENOMEM;
    }
    *out = c;
    return WD_OK;
}

int wd_destroy(wd_ctx* ctx) {
    if (!ctx) return WD_EINVAL;
    wd_graphs_clear(ctx);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    if (ctx->h_pinned) cudaFreeHost(ctx->h_pinned);
    for (cudaEvent_t e : ctx->prof_ev) cudaEventDestroy(e);
    delete ctx;
    return WD_OK;
}

int wd_set_option(wd_ctx* ctx, int key, int value) {
    if (!ctx) return WD_EINVAL;
    switch (key) {
        case WD_OPT_HOP32_SITES:
        case WD_OPT_HOP64_SITES:
            if (value < 0 || value > 1024) return wd_fail(ctx, WD_EINVAL, "sites per CTA out of range");
            break;
        case WD_OPT_HOP32_REGS:
        case WD_OPT_HOP64_REGS:
            if (value != 0 && (value < 32 || value > 255)) return wd_fail(ctx, WD_EINVAL, "register budget out of range");
            break;
        case WD_OPT_HOP_IMPL:
            if (value < 0 || value > 3) return wd_fail(ctx, WD_EINVAL, "hop implementation is 0, 1, 2 or 3");
            break;
        case WD_OPT_ALTERNATE_SWEEP:
        case WD_OPT_PAIRED:
        case WD_OPT_GRAPH:
        case WD_OPT_MERGE:
            if (value != 0 && value != 1) return wd_fail(ctx, WD_EINVAL, "this option is 0 or 1");
            break;
        case WD_OPT_HOP_ROWS:
            if (value < 0 || value > 1024) return wd_fail(ctx, WD_EINVAL, "rows per group out of range");
            break;
        case WD_OPT_SOLVER:
            if (value < 0 || value >= WD_SOLVER_N) return wd_fail(ctx, WD_EINVAL, "unknown solver");
            break;
        case WD_OPT_POLL_EVERY:
            if (value < 1 || value > 1024) return wd_fail(ctx, WD_EINVAL, "poll interval out of range");
            break;
        default:
            return wd_fail(ctx, WD_EINVAL, "unknown option");
    }
    ctx->opt[key] = value;
    wd_graphs_clear(ctx);   // captured launch shapes may depend on any of them
    return WD_OK;
}

int wd_get_option(const wd_ctx* ctx, int key, int* value) {
    if (!ctx || !value || key < 0 || key >= WD_OPT_N) return WD_EINVAL;
    *value = ctx->opt[key];
    return WD_OK;
}

int wd_profile(wd_ctx* ctx, int enable) {
    if (!ctx) return WD_EINVAL;
    if (ctx->prof_on != (enable != 0)) wd_graphs_clear(ctx);   // graphs with and without event nodes differ
    ctx->prof_on = enable != 0;
    return WD_OK;
}

int wd_profile_read(wd_ctx* ctx, double* ms, long long* count) {
    if (!ctx) return WD_EINVAL;
    if (!ms || !count) return wd_fail(ctx, WD_EINVAL, "null pointer");
    for (int k = 0; k < WD_PROF_N; ++k) { ms[k] = 0.0; count[k] = 0; }
    WD_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    for (size_t i = 0; i < ctx->prof_used; ++i) {
        float t = 0.f;
        WD_CUDA_CHECK(ctx, cudaEventElapsedTime(&t, ctx->prof_ev[2 * i], ctx->prof_ev[2 * i + 1]));
        ms[ctx->prof_cls[i]] += t;
        count[ctx->prof_cls[i]] += 1;
    }
    ctx->prof_used = 0;
    for (int k = 0; k < WD_PROF_N; ++k) {   // what the graph replays recorded (wd_solve.cu)
        ms[k] += ctx->prof_acc_ms[k];
        count[k] += ctx->prof_acc_cnt[k];
        ctx->prof_acc_ms[k] = 0.0;
        ctx->prof_acc_cnt[k] = 0;
    }
    return WD_OK;
}

int wd_site_order(wd_ctx* ctx, int order, const int tile[4]) {
    if (!ctx) return WD_EINVAL;
    if (ctx->have_ws) return wd_fail(ctx, WD_ESTATE, "wd_site_order must precede wd_set_workspace");
    if (order == WD_ORDER_LINEAR) {
        ctx->order = order;
    } else if (order == WD_ORDER_TILED) {
        if (!tile) return wd_fail(ctx, WD_EINVAL, "tile is null");
        for (int d = 0; d < 4; ++d)
            if (tile[d] < 1 || ctx->L[d] % tile[d]) return wd_fail(ctx, WD_EINVAL, "tile must divide dims");
        if (tile[0] & 1) return wd_fail(ctx, WD_EINVAL, "tile[0] must be even");
        ctx->order = order;
        for (int d = 0; d < 4; ++d) ctx->tile[d] = tile[d];
    } else {
        return wd_fail(ctx, WD_EINVAL, "unknown site order");
    }
    try {
        build_tables(ctx);
    } catch (const std::bad_alloc&) {
        return wd_fail(ctx, WD_ENOMEM, "site tables");
    }
    return WD_OK;
}

size_t wd_workspace_bytes(const wd_ctx* ctx) { return ctx ? ws_map(ctx).total : 0; }

int wd_set_workspace(wd_ctx* ctx, void* ws_dev, size_t bytes) {
    if (!ctx) return WD_EINVAL;
    if (!ws_dev) return wd_fail(ctx, WD_EINVAL, "workspace is null");
    if (((uintptr_t)ws_dev) & 255) return wd_fail(ctx, WD_EINVAL, "workspace must be 256-byte aligned");
    const WsMap m = ws_map(ctx);
    if (bytes < m.total) return wd_fail(ctx, WD_EINVAL, "workspace too small");
    wd_graphs_clear(ctx);
    char* w = (char*)ws_dev;
    ctx->ws = w;
    ctx->ws_bytes = bytes;
    ctx->d_site_of = (int32_t*)(w + m.site_of);
    ctx->d_nbr = (int32_t*)(w + m.nbr);
    for (int r = 0; r < 2; ++r) { ctx->d_U64[r] = (double*)(w + m.u64[r]); ctx->d_U32[r] = (float*)(w + m.u32[r]); }
    for (int r = 0; r < 2; ++r) ctx->d_U32P[r] = ctx->paired_ok ? (float*)(w + m.u32p[r]) : nullptr;
    ctx->d_scal = (double*)(w + m.scal);
    ctx->d_partials = (double*)(w + m.partials);
    ctx->partial_doubles = partial_doubles(ctx);
    ctx->d_totals = ctx->d_scal + 48 * WD_MAX_RHS;  // tail of the scalar block (kScalDoubles = 64 * WD_MAX_RHS)
    ctx->d_ticket = (unsigned int*)(w + m.ticket);
    ctx->d_solver = w + m.solver;
    ctx->solver_bytes = m.total - m.solver;
    WD_CUDA_CHECK(ctx, cudaMemcpyAsync(ctx->d_site_of, ctx->h_site_of.data(), sizeof(int32_t) * 2 * ctx->Vh,
                                       cudaMemcpyHostToDevice, ctx->stream));
    WD_CUDA_CHECK(ctx, cudaMemcpyAsync(ctx->d_nbr, ctx->h_nbr.data(), sizeof(int32_t) * 2 * ctx->Vh * WD_NDIR,
                                       cudaMemcpyHostToDevice, ctx->stream));
    WD_CUDA_CHECK(ctx, cudaMemsetAsync(ctx->d_ticket, 0, 256, ctx->stream));
    WD_CUDA_CHECK(ctx, cudaMemsetAsync(ctx->d_scal, 0, sizeof(double) * kScalDoubles, ctx->stream));
    WD_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));  // host tables may now change
    ctx->have_ws = true;
    ctx->have_gauge = false;
    return WD_OK;
}

int wd_set_gauge(wd_ctx* ctx, const double* U) {
    if (!ctx) return WD_EINVAL;
    if (!U) return wd_fail(ctx, WD_EINVAL, "gauge pointer is null");
    if (!ctx->have_ws) return wd_fail(ctx, WD_ESTATE, "wd_set_workspace first");
    int rc = wd_layout_gauge(ctx, U);
    if (rc == WD_OK) ctx->have_gauge = true;
    return rc;
}

size_t wd_native_bytes(const wd_ctx* ctx, int prec, int n_rhs) {
    if (!ctx || n_rhs < 0 || !wd_is_prec(prec) || (prec == WD_F32P && !ctx->paired_ok)) return 0;
    return 2 * wd_half_bytes(ctx, prec, n_rhs);
}

int wd_pack(wd_ctx* ctx, int prec, int n_rhs, const double* canon, void* native) {
    if (!ctx) return WD_EINVAL;
    if (!canon || !native || bad_n(ctx, n_rhs) || !wd_is_prec(prec))
        return wd_fail(ctx, WD_EINVAL, "wd_pack: bad argument");
    if (prec == WD_F32P && !ctx->paired_ok) return wd_fail(ctx, WD_EINVAL, "wd_pack: WD_F32P needs the row-major layout");
    if (!ctx->have_ws) return wd_fail(ctx, WD_ESTATE, "wd_set_workspace first");
    return wd_layout_pack(ctx, prec, n_rhs, canon, native);
}

int wd_unpack(wd_ctx* ctx, int prec, int n_rhs, const void* native, double* canon) {
    if (!ctx) return WD_EINVAL;
    if (!canon || !native || bad_n(ctx, n_rhs) || !wd_is_prec(prec))
        return wd_fail(ctx, WD_EINVAL, "wd_unpack: bad argument");
    if (prec == WD_F32P && !ctx->paired_ok) return wd_fail(ctx, WD_EINVAL, "wd_unpack: WD_F32P needs the row-major layout");
    if (!ctx->have_ws) return wd_fail(ctx, WD_ESTATE, "wd_set_workspace first");
    return wd_layout_unpack(ctx, prec, n_rhs, native, canon);
}

static int check_solver_params(wd_ctx* ctx, double tol, int max_outer, int max_inner, double inner_tol) {
    if (!(tol > 0.0) || max_outer < 1 || max_inner < 1 || !(inner_tol >= 0.0) || inner_tol >= 1.0)
        return wd_fail(ctx, WD_EINVAL, "bad solver parameters");
    return WD_OK;
}

static int check_op_args(wd_ctx* ctx, int op, int prec, int recon, int n_rhs, const void* a, const void* b) {
    if (!ctx) return WD_EINVAL;
    if (!a || !b || a == b) return wd_fail(ctx, WD_EINVAL, "null or aliased field pointer");
    if (bad_n(ctx, n_rhs)) return wd_fail(ctx, WD_EINVAL, "n_rhs out of range");
    if (op != WD_OP_D && op != WD_OP_DDAG) return wd_fail(ctx, WD_EINVAL, "bad op");
    if (!wd_is_prec(prec)) return wd_fail(ctx, WD_EINVAL, "bad precision");
    if (prec == WD_F32P && !ctx->paired_ok) return wd_fail(ctx, WD_EINVAL, "WD_F32P needs the row-major layout");
    if (recon != WD_LINK18 && recon != WD_LINK12) return wd_fail(ctx, WD_EINVAL, "bad link form");
    if (!ctx->have_gauge) return wd_fail(ctx, WD_ESTATE, "wd_set_gauge first");
    return WD_OK;
}

int wd_apply(wd_ctx* ctx, int op, int prec, int recon, int n_rhs, const void* in, void* out) {
    int rc = check_op_args(ctx, op, prec, recon, n_rhs, in, out);
    if (rc) return rc;
    const size_t hb = wd_half_bytes(ctx, prec, n_rhs);
    const char* i = (const char*)in;
    char* o = (char*)out;
    // out_p = in_p - kappa H_{p,1-p} in_{1-p}   (D = 1 - kappa H; reading R4)
    for (int p = 0; p < 2; ++p) {
        rc = wd_hop_launch(ctx, prec, recon, op == WD_OP_DDAG, n_rhs, p, i + (1 - p) * hb, o + p * hb, i + p * hb,
                           1.0, -ctx->kappa);
        if (rc) return rc;
    }
    return WD_OK;
}

int wd_hop(wd_ctx* ctx, int op, int prec, int recon, int n_rhs, int out_parity, const void* in, void* out) {
    int rc = check_op_args(ctx, op, prec, recon, n_rhs, in, out);
    if (rc) return rc;
    if (out_parity != 0 && out_parity != 1) return wd_fail(ctx, WD_EINVAL, "bad parity");
    return wd_hop_launch(ctx, prec, recon, op == WD_OP_DDAG, n_rhs, out_parity, in, out, nullptr, 0.0, 1.0);
}

int wd_solve_block(wd_ctx* ctx, int op, int n_rhs, const double* Phi, double* X, double tol, int max_outer,
                   int max_inner, double inner_tol, int recon, wd_solve_info* info) {
    int rc = check_op_args(ctx, op, WD_F64, recon, n_rhs, Phi, X);
    if (rc) return rc;
    rc = check_solver_params(ctx, tol, max_outer, max_inner, inner_tol);
    if (rc) return rc;
    return wd_solve_impl(ctx, op == WD_OP_DDAG, n_rhs, Phi, X, tol, max_outer, max_inner, inner_tol, recon, info);
}

int wd_force(wd_ctx* ctx, int n_rhs, const double* X, const double* Y, double* F) {
    if (!ctx) return WD_EINVAL;
    if (!X || !Y || !F) return wd_fail(ctx, WD_EINVAL, "null pointer");
    if (bad_n(ctx, n_rhs)) return wd_fail(ctx, WD_EINVAL, "n_rhs out of range");
    if (!ctx->have_gauge) return wd_fail(ctx, WD_ESTATE, "wd_set_gauge first");
    return wd_force_impl(ctx, n_rhs, X, Y, F);
}

static int md_force_host_common(wd_ctx* ctx, int n_rhs, const double* U_host, const double* Phi_host, double* F_host,
                                double tol, int max_outer, int max_inner, double inner_tol, int recon,
                                wd_solve_info* info2) {
    if (!ctx) return WD_EINVAL;
    if (!Phi_host || !F_host) return wd_fail(ctx, WD_EINVAL, "null pointer");
    if (bad_n(ctx, n_rhs)) return wd_fail(ctx, WD_EINVAL, "n_rhs out of range");
    if (recon != WD_LINK18 && recon != WD_LINK12) return wd_fail(ctx, WD_EINVAL, "bad link form");
    if (!U_host && !ctx->have_gauge) return wd_fail(ctx, WD_ESTATE, "wd_set_gauge first");
    if (U_host && !ctx->have_ws) return wd_fail(ctx, WD_ESTATE, "wd_set_workspace first");
    int rcp = check_solver_params(ctx, tol, max_outer, max_inner, inner_tol);
    if (rcp) return rcp;
    // staging lives at the END of the solver scratch (sized for max_rhs in wd_solver_scratch_bytes)
    const size_t full = wd_align_up(2 * wd_half_bytes(ctx, WD_F64, ctx->max_rhs));
    const size_t fbytes = wd_align_up(sizeof(double) * 4 * ctx->V * 18);
    char* end = ctx->d_solver + ctx->solver_bytes;
    double* dF = (double*)(end - fbytes);
    double* dY = (double*)(end - fbytes - full);
    double* dX = (double*)(end - fbytes - 2 * full);
    double* dPhi = (double*)(end - fbytes - 3 * full);
    double* dCanon = (double*)(end - fbytes - 4 * full);
    if (U_host) {   // a0: the canonical links go through dF (same size), which is cleared afterwards
        WD_CUDA_CHECK(ctx, cudaMemcpyAsync(dF, U_host, sizeof(double) * 4 * ctx->V * 18, cudaMemcpyHostToDevice, ctx->stream));
        int rcg = wd_layout_gauge(ctx, dF);
        if (rcg) return rcg;
        ctx->have_gauge = true;
    }
    const size_t cbytes = sizeof(double) * 24 * ctx->V * n_rhs;
    WD_CUDA_CHECK(ctx, cudaMemcpyAsync(dCanon, Phi_host, cbytes, cudaMemcpyHostToDevice, ctx->stream));
    int rc = wd_layout_pack(ctx, WD_F64, n_rhs, dCanon, dPhi);
    if (rc) return rc;
    WD_CUDA_CHECK(ctx, cudaMemsetAsync(dF, 0, sizeof(double) * 4 * ctx->V * 18, ctx->stream));
    const double itol = inner_tol;
    rc = wd_md_force_impl(ctx, WD_ACTION_FULL, n_rhs, dPhi, dX, dY, dF, nullptr, dCanon, tol, max_outer, max_inner, itol,
                          recon, info2);
    if (rc != WD_OK && rc != WD_ENOCONV) return rc;
    WD_CUDA_CHECK(ctx, cudaMemcpyAsync(F_host, dF, sizeof(double) * 4 * ctx->V * 18, cudaMemcpyDeviceToHost, ctx->stream));
    WD_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    return rc;
}

int wd_md_force_host(wd_ctx* ctx, int n_rhs, const double* Phi_host, double* F_host, double tol, int max_outer,
                     int max_inner, double inner_tol, int recon, wd_solve_info* info2) {
    return md_force_host_common(ctx, n_rhs, nullptr, Phi_host, F_host, tol, max_outer, max_inner, inner_tol, recon, info2);
}

int wd_md_force_host_gauge(wd_ctx* ctx, int n_rhs, const double* U_host, const double* Phi_host, double* F_host, double tol,
                           int max_outer, int max_inner, double inner_tol, int recon, wd_solve_info* info2) {
    if (ctx && !U_host) return wd_fail(ctx, WD_EINVAL, "null pointer");
    return md_force_host_common(ctx, n_rhs, U_host, Phi_host, F_host, tol, max_outer, max_inner, inner_tol, recon, info2);
}

int wd_refresh(wd_ctx* ctx, int variant, int n_rhs, const double* eta, double* phi) {
    int rc = check_op_args(ctx, WD_OP_D, WD_F64, WD_LINK18, n_rhs, eta, phi);
    if (rc) return rc;
    if (variant != WD_ACTION_FULL && variant != WD_ACTION_EO) return wd_fail(ctx, WD_EINVAL, "bad action variant");
    return wd_refresh_impl(ctx, variant, n_rhs, eta, phi);
}

int wd_action(wd_ctx* ctx, int n_rhs, int parity_sel, const double* X, double* S_host) {
    if (!ctx) return WD_EINVAL;
    if (!X || !S_host) return wd_fail(ctx, WD_EINVAL, "null pointer");
    if (bad_n(ctx, n_rhs)) return wd_fail(ctx, WD_EINVAL, "n_rhs out of range");
    if (parity_sel < WD_PARITY_EVEN || parity_sel > WD_PARITY_BOTH) return wd_fail(ctx, WD_EINVAL, "bad parity selection");
    if (!ctx->have_ws) return wd_fail(ctx, WD_ESTATE, "wd_set_workspace first");
    return wd_action_impl(ctx, n_rhs, parity_sel, X, S_host);
}

int wd_set_residual_history(wd_ctx* ctx, double* hist_dev, int capacity) {
    if (!ctx) return WD_EINVAL;
    if (capacity < 0 || (hist_dev && capacity == 0) || ((size_t)hist_dev & 7) != 0)
        return wd_fail(ctx, WD_EINVAL, "wd_set_residual_history: bad capacity or misaligned buffer");
    ctx->d_hist = capacity > 0 ? hist_dev : nullptr;
    ctx->hist_cap = ctx->d_hist ? capacity : 0;
    wd_graphs_clear(ctx);   // the captured iteration blocks carry the pointer
    return WD_OK;
}

int wd_inner_plan(const wd_ctx* ctx, int n_rhs, int recon, int* plan_host) {
    if (!ctx || !plan_host) return WD_EINVAL;
    if (bad_n(ctx, n_rhs) || (recon != WD_LINK18 && recon != WD_LINK12)) return WD_EINVAL;
    bool paired, merged;
    wd_inner_forms(ctx, recon, n_rhs, &paired, &merged);
    plan_host[WD_PLAN_HOP_KERNEL] = paired ? WD_HOP_KERNEL_ZMARCH : wd_hop_kernel_for(ctx, WD_F32, recon, n_rhs);
    plan_host[WD_PLAN_MERGED] = merged ? 1 : 0;
    plan_host[WD_PLAN_PAIRED] = paired ? 1 : 0;
    plan_host[WD_PLAN_KERNELS_PER_ITER] = merged ? 6 : 7;
    return WD_OK;
}

int wd_project_parity(wd_ctx* ctx, int prec, int n_rhs, int parity, void* native) {
    if (!ctx) return WD_EINVAL;
    if (!native || bad_n(ctx, n_rhs) || (prec != WD_F64 && prec != WD_F32) || (parity != 0 && parity != 1))
        return wd_fail(ctx, WD_EINVAL, "wd_project_parity: bad argument");
    return wd_project_parity_impl(ctx, prec, n_rhs, parity, native);
}

int wd_md_force(wd_ctx* ctx, int variant, int n_rhs, const double* Phi, double* X, double* Y, double* F, double* S_host,
                double tol, int max_outer, int max_inner, double inner_tol, int recon, wd_solve_info* info2) {
    int rc = check_op_args(ctx, WD_OP_D, WD_F64, recon, n_rhs, Phi, X);
    if (rc) return rc;
    if (!Y || !F || Y == X || (const double*)Y == Phi) return wd_fail(ctx, WD_EINVAL, "null or aliased field pointer");
    if (variant != WD_ACTION_FULL && variant != WD_ACTION_EO) return wd_fail(ctx, WD_EINVAL, "bad action variant");
    rc = check_solver_params(ctx, tol, max_outer, max_inner, inner_tol);
    if (rc) return rc;
    // scratch for the projected right-hand sides of the even/odd variant: the host path's canonical staging block
    const size_t full = wd_align_up(2 * wd_half_bytes(ctx, WD_F64, ctx->max_rhs));
    const size_t fbytes = wd_align_up(sizeof(double) * 4 * ctx->V * 18);
    double* tmp = (double*)(ctx->d_solver + ctx->solver_bytes - fbytes - 4 * full);
    return wd_md_force_impl(ctx, variant, n_rhs, Phi, X, Y, F, S_host, tmp, tol, max_outer, max_inner,
                            inner_tol, recon, info2);
}

}  // extern "C"
