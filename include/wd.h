/* wd.h -- C ABI of the B200 (sm_100a) blocked Wilson-Dirac solve + fermion force library.
 *
 * What it computes (arxiv/paper_1009_5169, "Algorithm 2", eq. 2.3):
 *     2: solve D X = Phi          X  = D^-1 Phi            (N_f/2 columns at once)
 *     3: solve D^dag Y = X        Y  = D^dag^-1 X
 *     5: F_mu = F_mu + f[x_i, y_i]   for every column i
 * with D the Wilson-Dirac operator on a lattice with Schroedinger-functional (Dirichlet) time
 * boundaries.  The paper fixes neither the normalisation of D, the gamma basis, the
 * SF convention nor f[x,y]; the readings used are listed in DESIGN.md section 2:
 *     D = 1 - kappa H,
 *     (H psi)(x) = sum_mu (1-gamma_mu) U_mu(x) psi(x+mu) + (1+gamma_mu) U_mu(x-mu)^dag psi(x-mu),
 *     D^dag: gamma_mu -> -gamma_mu;   SF: psi(t=0) = psi(t=T) = 0, T slices stored (t = 0..T-1),
 *     f[x,y]_mu(s) = 2 kappa TA[ U_mu(s) W ],  TA(M) = (M - M^dag)/2 - tr(M - M^dag)/6,
 *     W = sum_spin x(s+mu) (x) ((1-gamma_mu) y(s))^dag + ((1+gamma_mu) y(s+mu)) (x) x(s)^dag.
 *
 * Conventions common to every call
 *   - Every function returns an int: WD_OK (0) or a negative WD_E* code.  Nothing throws or aborts
 *     across this boundary.  wd_last_error(ctx) gives a text for the last failure on that context.
 *   - Pointers named *_dev are DEVICE pointers (cudaMalloc'ed by the caller, e.g. a torch tensor's
 *     data_ptr()); pointers named *_host are HOST pointers.  The caller owns every buffer it
 *     passes; the library owns only the context and never allocates device memory after
 *     wd_set_workspace (all its scratch is carved from the caller's workspace).
 *   - All work is enqueued on the CUDA stream given to wd_create.  wd_apply, wd_pack, wd_unpack,
 *     wd_force and wd_set_gauge do not synchronise.  wd_solve_block synchronises the stream to
 *     read convergence scalars.  The *_host entry points synchronise before returning.
 *   - dims = (Lx, Ly, Lz, T), all even, >= 2 (>= 4 in T for WD_BC_SF).  mu = 0,1,2,3 = x,y,z,t.
 *
 * Layouts
 *   CANONICAL (fp64, what a user holds):
 *     gauge / force  double [mu=4][T][Lz][Ly][Lx][3][3][2]    row-major colour matrix, (re,im)
 *     spinor block   double [n_rhs][T][Lz][Ly][Lx][4][3][2]   spin, colour, (re,im)
 *   NATIVE (what the kernels read; produced by wd_pack, consumed by wd_unpack):
 *     sites are split by parity (x+y+z+t) mod 2 (even = 0) and numbered 0..V/2-1 inside a parity
 *     in the context's site order (wd_site_order); the V/2 sites of a parity are cut into layout blocks of
 *     RB consecutive sites (site h = b*RB + o) and a full-lattice block of n_rhs spinors is
 *       fp64:  double2 [parity=2][b][k=12][o=RB][n_rhs]    k = spin*3+colour, one complex per double2
 *       fp32:  float4  [parity=2][b][c=6 ][o=RB][n_rhs]    complex 2c and 2c+1 per float4
 *     i.e. structure-of-arrays, site-major / RHS-minor, 128-bit elements.  RB = Lx/2 (a block is one
 *     lattice row with all its chunks: what the staged hopping kernel copies in bulk) for the linear site
 *     order when Lx/2 is even and max_rhs >= 3, else RB = V/2 (plain chunk-major).  The layout is an
 *     internal matter of the library: wd_pack / wd_unpack are the way in and out.  wd_native_bytes gives
 *     the size.  In SF mode the t=0 slice is stored and is zero in every native field the library
 *     produces; wd_pack writes zeros there whatever the canonical input holds.
 */
#ifndef WD_H
#define WD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wd_ctx wd_ctx; /* opaque; created by wd_create, freed by wd_destroy */

enum { WD_OK = 0, WD_EINVAL = -1, WD_ENOMEM = -2, WD_ECUDA = -3, WD_ENOCONV = -4, WD_ESTATE = -5 };
enum { WD_BC_PERIODIC = 0, WD_BC_SF = 1 }; /* time direction; space is always periodic, theta=0 */
enum { WD_OP_D = 0, WD_OP_DDAG = 1 };
/* WD_F32P: fp32 in the x-paired native form "P32" -- two sites of a lattice row (Lx/4 apart within their parity) share
 * every 128-bit element, one complex number each, so that one thread works on both with the packed fp32 instructions of
 * sm_100 (csrc/wd_f2.cuh).  It is the form the fp32 inner solver computes in (wd_solve_block) and is
 * accepted by wd_native_bytes, wd_pack, wd_unpack, wd_hop and wd_apply so that it can be tested and timed on its own;
 * results are bit for bit those of WD_F32.  Needs the row-major layout (linear site order, Lx/2 even, max_rhs >= 3) and
 * a (lattice, n_rhs) shape the z-march hop kernel serves; elsewhere those calls return WD_EINVAL and the solver
 * computes in WD_F32. */
enum { WD_F64 = 0, WD_F32 = 1, WD_F32P = 2 };
enum { WD_LINK18 = 0, WD_LINK12 = 1 }; /* 18 reals per link, or rows 1-2 only */
enum { WD_ORDER_LINEAR = 0, WD_ORDER_TILED = 1 };
enum { WD_ACTION_FULL = 0, WD_ACTION_EO = 1 };   /* pseudo-fermion action on D (eq. 2.2) or on the even/odd Schur complement */
enum { WD_PARITY_EVEN = 0, WD_PARITY_ODD = 1, WD_PARITY_BOTH = 2 };

#define WD_MAX_RHS 16

/* Filled by wd_solve_block (all host memory, owned by the caller). */
typedef struct wd_solve_info {
    int    n_rhs;
    int    outer_steps;               /* fp64 defect-correction steps taken (inner solver calls)     */
    int    inner_iters_total;         /* fp32 BiCGStab iterations summed over the outer steps         */
    int    converged;                 /* 1 if every column met tol                                    */
    double relres[WD_MAX_RHS];        /* final TRUE fp64 residual |phi_i - A x_i| / |phi_i|            */
    double bnorm[WD_MAX_RHS];         /* |phi_i|                                                      */
    double seconds;                   /* host wall time of the call (includes its synchronisations)   */
} wd_solve_info;

/* Create a context for a lattice (problem statement: "SF setup ... Wilson quarks",
 * kappa = hopping parameter).  time_bc = WD_BC_SF gives the Dirichlet time boundaries.  max_rhs
 * (1..WD_MAX_RHS) bounds n_rhs of every later call and sizes the workspace.  cuda_stream is a
 * cudaStream_t (NULL = legacy default stream).  Errors: WD_EINVAL (null, odd or too small dims,
 * kappa not finite, max_rhs out of range), WD_ECUDA (no device), WD_ENOMEM (host). */
int wd_create(wd_ctx** out, const int dims[4], double kappa, int time_bc, int max_rhs, void* cuda_stream);
int wd_destroy(wd_ctx* ctx);

/* Choose how sites are numbered inside a parity (affects only the native layout, hence speed):
 * WD_ORDER_LINEAR: x/2 fastest, then y, z, t.  WD_ORDER_TILED: blocks of tile[] = (bx,by,bz,bt)
 * full-lattice sites are contiguous (each must divide the matching dim; bx even).  Must be
 * called before wd_set_workspace; default is WD_ORDER_LINEAR.  Errors: WD_EINVAL, WD_ESTATE. */
int wd_site_order(wd_ctx* ctx, int order, const int tile[4]);

/* Launch tunables (speed only, never results).  Keys:
 *   WD_OPT_HOP32_SITES / WD_OPT_HOP64_SITES  sites per CTA of the fp32 / fp64 hopping kernel (a CTA has
 *       sites * n_rhs threads, halved until <= 1024).  0 (default) = chosen from n_rhs; else 1..1024.
 *   WD_OPT_HOP32_REGS / WD_OPT_HOP64_REGS    register budget per thread: picks among the compiled
 *       variants (fp32: 64, 128; fp64: 128, 168), clamped so that one CTA fits an SM.  0 (default) = chosen from n_rhs.
 *   WD_OPT_HOP_IMPL     which hopping kernel serves a launch.  The two staged kernels (persistent CTAs, producer warps
 *       feeding shared memory with cp.async.bulk + mbarrier, consumer warps) need the row-major native layout (linear
 *       site order, Lx/2 even) and n_rhs >= 3; everything else goes to the register kernel.
 *       2 (default): fp32: the z-march kernel (sliding window of three lattice planes) or, where its step would be
 *          small and the rows long, the row-group ring kernel (csrc/wd_hop_zm.cu wd_hop_zm_preferred); fp64: the ring kernel.
 *       3: the z-march kernel wherever it can run at all (fp32).
 *       1: the ring kernel.
 *       0: always the register kernel (one thread per site and column, operands loaded straight into registers).
 *       The register and z-march kernels agree bit for bit; the ring kernel adds the eight directions in another order.
 *   WD_OPT_HOP_ROWS     staged kernel: upper bound on the lattice rows (consecutive in y) one CTA works on at a
 *       time; 0 (default) = as many as the thread and shared-memory budgets allow.  Fewer rows = smaller
 *       units, more ring slots (deeper prefetch), fewer consumer warps.
 *   WD_OPT_ALTERNATE_SWEEP  1 (default): consecutive kernels of the inner solver sweep the vectors in opposite
 *       directions, so that what one kernel wrote last is still in L2 when the next reads it first; 0: off.
 *   WD_OPT_POLL_EVERY   inner iterations enqueued between two convergence polls of the solver (>= 1).
 *   WD_OPT_SOLVER       the route wd_solve_block (and everything built on it) takes to the SAME result X = A^-1 Phi
 *       within tol; iteration counts differ.
 *       WD_SOLVER_DC_F32 (default): fp64 defect correction around an fp32-storage BiCGStab (reading R11).
 *       WD_SOLVER_RELIABLE_H16: one continuous BiCGStab sequence per column with the vectors STORED in 16 bits
 *       (fp16 mantissas + one fp32 scale per spinor, arithmetic in fp32) and fp64 reliable updates in place of
 *       restarts ("tuning techniques described in [4]"); inner_tol is then the
 *       reliable-update threshold delta (0 = default 0.01), max_outer bounds the number of updates and max_inner the
 *       total number of iterations ENQUEUED (between the moment a column asks for an update and the next poll, up to
 *       WD_OPT_POLL_EVERY - 1 enqueued iterations are no-ops; info.inner_iters_total counts the ones that did work).
 *       Needs the z-march hop kernel with 16-bit operands (linear site order, Lx/2 even, n_rhs >= 3, Lx/2 * n_rhs a
 *       multiple of 4 and at most 384, the consumer threads of one CTA); elsewhere the default solver runs.
 *       WD_SOLVER_GL_FLEX: the paper's case D1 (Table 1): fp64 Global BiCGStab (one alpha, beta, omega for the
 *       whole block, Frobenius inner products) in flexible form, preconditioned by the fp32 BiCGStab per column;
 *       max_outer bounds its iterations (two preconditioner calls each), info.outer_steps counts preconditioner calls.
 *       WD_SOLVER_GL_F64: case B, the same without preconditioner (all fp64; info.inner_iters_total = its iterations);
 *       there being no inner solver, max_inner bounds its iterations (as for WD_SOLVER_BL_F64) and max_outer is unused.
 *       These three blocked solvers stop on the recursive residual, then compute the true one (which info.relres
 *       reports) and restart from it for as long as a column misses tol and iterations are left.
 *       WD_SOLVER_BL_F64: case C, fp64 Block BiCGStab (ref. [7] of the paper): n_rhs x n_rhs coefficient matrices from the
 *       Gram matrices of the block vectors, one Krylov space shared by the columns; max_inner bounds its iterations.
 *       The n x n systems need a block of full rank: with a zero column, two equal columns, or on a breakdown of the
 *       recurrence (pivot below 1e-13 of the largest Gram entry) the iteration freezes and the default solver
 *       (WD_SOLVER_DC_F32) does the solve instead, with max_outer and max_inner as given.
 *   WD_OPT_PAIRED       1: the fp32 inner solver computes in the x-paired form WD_F32P (two sites per thread, packed
 *       fp32 instructions) wherever the z-march hop kernel serves the shape; 0 (default): plain WD_F32.  Same iterates
 *       up to the summation order of the inner products.  (Measured at 24^4, n_rhs = 5: 64 us against 59 us per hop --
 *       the hop is bound by shared-memory bandwidth, which pairing does not change, and has half the warps to hide
 *       latency with.)
 *   WD_OPT_GRAPH        1 (default): the fp32 inner solver replays each block of WD_OPT_POLL_EVERY iterations (7 kernels
 *       each, plus the read-back of the convergence flag) as one CUDA graph, captured the second time a (operator, n_rhs,
 *       link form) combination is solved; 0: plain stream launches.  Identical results; off while wd_profile is on.
 *   WD_OPT_MERGE        1 (default): the fp32 inner solver folds the p-update of iteration k+1 into the x,r-update of
 *       iteration k (one 8-stream kernel instead of a 7- and a 4-stream one: 23 instead of 25 vector passes per
 *       iteration, 6 instead of 7 kernels); the rho it needs comes from the second hop's epilogue as
 *       <rt,s> - omega <rt,t>.  Where the z-march hop kernel serves the shape; 0: the textbook order.  The iterates
 *       agree to rounding, the result to tol.
 * Errors: WD_EINVAL (null, unknown key, value out of range). */
enum { WD_OPT_HOP32_SITES = 0, WD_OPT_HOP64_SITES = 1, WD_OPT_HOP32_REGS = 2, WD_OPT_HOP64_REGS = 3,
       WD_OPT_POLL_EVERY = 4, WD_OPT_HOP_IMPL = 5, WD_OPT_ALTERNATE_SWEEP = 6, WD_OPT_HOP_ROWS = 7, WD_OPT_SOLVER = 8,
       WD_OPT_PAIRED = 9, WD_OPT_GRAPH = 10, WD_OPT_MERGE = 11, WD_OPT_N = 12 };
/* values of WD_OPT_SOLVER */
enum { WD_SOLVER_DC_F32 = 0, WD_SOLVER_RELIABLE_H16 = 1, WD_SOLVER_GL_FLEX = 2, WD_SOLVER_GL_F64 = 3, WD_SOLVER_BL_F64 = 4,
       WD_SOLVER_N = 5 };
int wd_set_option(wd_ctx* ctx, int key, int value);
int wd_get_option(const wd_ctx* ctx, int key, int* value_host);

/* Scratch memory: the caller allocates wd_workspace_bytes(ctx) bytes of device memory (256-byte
 * aligned) and hands it over; it must stay valid until wd_destroy.  wd_set_workspace uploads the
 * site tables.  Errors: WD_EINVAL (null, too small, misaligned), WD_ECUDA. */
size_t wd_workspace_bytes(const wd_ctx* ctx);
int    wd_set_workspace(wd_ctx* ctx, void* ws_dev, size_t bytes);

/* Gauge ingest (hot-path step a0): canonical fp64 links -> the library's native fp64 and fp32
 * copies, each in 18-real and 12-real form ("single-precision coefficient matrix D on the GPUs",
 * PAPER.md:84; "3rd column ... dropped ... reconstructed on the fly").  The canonical
 * buffer is not referenced after the enqueued kernels finish.  Errors: WD_ESTATE (no workspace). */
int wd_set_gauge(wd_ctx* ctx, const double* U_canon_dev);

/* Bytes of a native full-lattice block of n_rhs spinors in precision prec (WD_F64 / WD_F32). */
size_t wd_native_bytes(const wd_ctx* ctx, int prec, int n_rhs);

/* canonical fp64 block [n_rhs][T][Lz][Ly][Lx][4][3][2]  <->  native block of precision prec. */
int wd_pack(wd_ctx* ctx, int prec, int n_rhs, const double* canon_dev, void* native_dev);
int wd_unpack(wd_ctx* ctx, int prec, int n_rhs, const void* native_dev, double* canon_dev);

/* The operator of the linear systems of Algorithm 2 ("solve D X = Phi", "solve D^dag Y = X"; Wilson
 * quarks; the form of D is DESIGN.md reading R4, D^dag R5): out = D in (op = WD_OP_D) or D^dag in (WD_OP_DDAG) on a native full-lattice block, all n_rhs
 * columns in one pass per output parity (two launches of the hopping kernel with the diagonal
 * term fused).  prec picks fp64 or fp32 arithmetic and storage, recon the link form.  in and out
 * must not overlap.  Errors: WD_ESTATE (no gauge), WD_EINVAL (n_rhs, enums, null). */
int wd_apply(wd_ctx* ctx, int op, int prec, int recon, int n_rhs, const void* in_native_dev, void* out_native_dev);

/* The bare hopping term on one output parity (hot-path step a2; the kernel inside the paper's single-precision GPU
 * solver, whose even/odd form PAPER.md:74 names: D = 1 - kappa H), exposed for measurement:
 * out[out_parity] = H in[1-out_parity] ("dslash").  in/out are native HALF-lattice blocks, i.e.
 * [k or c][V/2][n_rhs] (half of wd_native_bytes).  Same errors as wd_apply. */
int wd_hop(wd_ctx* ctx, int op, int prec, int recon, int n_rhs, int out_parity, const void* in_half_dev, void* out_half_dev);

/* Blocked solve (Algorithm 2 lines 2-3): A X = Phi with A = D (WD_OP_D) or D^dag
 * (WD_OP_DDAG), Phi and X native fp64 full-lattice blocks (X may not alias Phi).  Route: site
 * even/odd preconditioning, fp64 defect-correction outer loop around an fp32
 * BiCGStab run in lock-step over the columns with per-column scalars.  Stops
 * when every column has |phi_i - A x_i| <= tol |phi_i| in fp64 (true residual), or after
 * max_outer outer steps of at most max_inner inner iterations each; inner_tol (0 = default 3e-7)
 * is the relative reduction asked of each inner call; recon picks the inner (fp32) link form,
 * the fp64 outer operator always uses 18 reals.  Returns WD_ENOCONV if tol was not met: X then
 * holds the best iterate and info is still filled.  info may be NULL. */
int wd_solve_block(wd_ctx* ctx, int op, int n_rhs, const double* Phi_native_dev, double* X_native_dev,
                   double tol, int max_outer, int max_inner, double inner_tol, int recon,
                   wd_solve_info* info);

/* Force accumulation (Algorithm 2 lines 4-6): F += sum_i f[x_i, y_i] with X, Y
 * native fp64 full-lattice blocks and F canonical fp64 [mu][T][Lz][Ly][Lx][3][3][2].  F is
 * ACCUMULATED ("F_mu = F_mu + f[x_i,y_i]"); the caller zeroes it. */
int wd_force(wd_ctx* ctx, int n_rhs, const double* X_native_dev, const double* Y_native_dev, double* F_canon_dev);

/* One whole MD force evaluation from HOST buffers (Algorithm 2 as a single call): copies the
 * canonical Phi to the device, packs, solves D X = Phi and D^dag Y = X, accumulates the force
 * into a zeroed device buffer and copies it to F_canon_host (overwritten, not accumulated).
 * Staging buffers come from the workspace.  info[0], info[1] (nullable) describe the two solves.
 * Synchronises.  Phi_canon_host/F_canon_host should be pinned for full copy bandwidth. */
int wd_md_force_host(wd_ctx* ctx, int n_rhs, const double* Phi_canon_host, double* F_canon_host,
                     double tol, int max_outer, int max_inner, double inner_tol, int recon,
                     wd_solve_info* info2);

/* One whole MD force evaluation from HOST buffers INCLUDING the gauge field (the links change between force
 * evaluations of a trajectory): copies the canonical U (4 V 18 doubles) and Phi to the device, runs the
 * gauge ingest (hot-path step a0) and then everything wd_md_force_host does.  U_canon_host should be pinned. */
int wd_md_force_host_gauge(wd_ctx* ctx, int n_rhs, const double* U_canon_host, const double* Phi_canon_host,
                           double* F_canon_host, double tol, int max_outer, int max_inner, double inner_tol, int recon,
                           wd_solve_info* info2);

/* The steps either side of the path in a molecular-dynamics step (PAPER.md:33-40 eq. 2.1-2.2, :60, :74).
 *
 * wd_refresh: pseudo-fermion heat bath.  variant = WD_ACTION_FULL: phi = D eta on the full lattice (then
 *   S = sum_i |D^-1 phi_i|^2 = sum_i |eta_i|^2).  WD_ACTION_EO: the pseudo-fermions live on the even sites and the
 *   action is written on Dhat = 1 - kappa^2 H_eo H_oe (the even/odd-preconditioned operator):
 *   phi_e = Dhat eta_e, phi_o = 0 (the odd half of eta is ignored).  eta, phi: native fp64 full-lattice blocks, no overlap.
 * wd_action: S_host[i] = |x_i|^2 over the sites selected by parity_sel (WD_PARITY_BOTH for the full action with
 *   x = D^-1 phi; WD_PARITY_EVEN for the even/odd variant); one fused fp64 norm kernel, synchronises.
 * wd_project_parity: native = P_parity native (the other parity's sites are zeroed), in place.
 * wd_md_force: Algorithm 2 on DEVICE-resident native fields: X = A^-1 Phi, Y = A^dag^-1 X',
 *   F += sum_i f[x_i, y_i], S_host[i] (nullable) = action per column.  WD_ACTION_FULL: A = D, X' = X.
 *   WD_ACTION_EO: right-hand sides P_e Phi and X' = P_e X, i.e. x_e = Dhat^-1 phi_e, X = (x_e, kappa H_oe x_e) and Y
 *   likewise, with the same force functional (reading R16).  X, Y: native fp64 outputs; F canonical,
 *   accumulated; info2[0], info2[1] (nullable) describe the two solves.  Solver parameters as wd_solve_block.
 * Errors: WD_EINVAL (null, n_rhs, enums), WD_ESTATE (no gauge), WD_ENOCONV. */
int wd_refresh(wd_ctx* ctx, int variant, int n_rhs, const double* eta_native_dev, double* phi_native_dev);
int wd_action(wd_ctx* ctx, int n_rhs, int parity_sel, const double* X_native_dev, double* S_host);
int wd_project_parity(wd_ctx* ctx, int prec, int n_rhs, int parity, void* native_dev);
int wd_md_force(wd_ctx* ctx, int variant, int n_rhs, const double* Phi_native_dev, double* X_native_dev,
                double* Y_native_dev, double* F_canon_dev, double* S_host, double tol, int max_outer, int max_inner,
                double inner_tol, int recon, wd_solve_info* info2);

/* The action without a context, a workspace or any allocation: S_dev[i] = sum over the block of |x_i|^2, i.e. what
 * wd_action computes (eq. 2.2; the number the Metropolis step of PAPER.md:60 needs), for callers that
 * cannot allocate device memory -- a lattice code that has given the whole card to its own field arena, or code that
 * must not stall other streams (cudaMalloc and cudaFree synchronise the device).  wd_action needs a context whose
 * workspace the caller has to cudaMalloc; this call needs neither.  It calls no cudaMalloc, cudaFree, cudaMallocHost
 * or any other allocating routine, creates no stream or event, and does not synchronise.
 *   X_native_dev  DEVICE, read: n_complex consecutive complex numbers (double2) of a native fp64 block, RHS-minor,
 *                 starting at a multiple of n_rhs complex numbers -- a whole block (wd_native_bytes / 16 numbers), or one
 *                 parity half of it (the first half is the even sites, the second the odd ones).  16-byte aligned.
 *   S_dev         DEVICE, written: n_rhs doubles, overwritten (not accumulated) by the kernel.  The result is there
 *                 when the work enqueued on cuda_stream has finished; nothing is copied to the host.
 *   cuda_stream   a cudaStream_t of the CURRENT device (NULL = legacy default stream).  X and S must be memory of
 *                 that device too (checked).
 * Scratch: the per-block partial sums and a ticket counter live in a fixed __device__ array inside the library,
 * WD_STATIC_SCRATCH_BYTES (2 MiB + 256 B) that every GPU which loads libwd.so holds until the process exits.  Its size
 * bounds the input: n_complex / n_rhs <= WD_STATIC_MAX_ROWS (2^25; a 24^4 block has 4.0e6 such rows for any n_rhs, a
 * 40^4 block 3.1e7); beyond that the call returns WD_EINVAL and wd_action_static_error() says so -- use wd_action.
 * Sharing: every call on a device uses the same array, which keeps what the previous call left in it; the call
 * clears the one word that must start at zero (stream-ordered, before its kernel).  Calls enqueued on ONE stream are
 * therefore safe back to back; two calls that can overlap on the GPU (different streams or threads, same device)
 * race on the array and give wrong sums -- order them with an event.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, once per device, with that
 * device current), which can make the driver load the library's kernels; make that first call at set-up time, before
 * any stream capture is begun.
 * The sum is fp64 and its order depends only on (n_rhs, n_complex), not on the GPU: the same input gives the same
 * bits everywhere (wd_action's order depends on the SM count; the two agree to rounding, ~1e-15 relative).
 * Errors: WD_EINVAL (n_rhs outside 1..WD_MAX_RHS, null or misaligned pointer, n_complex zero or not a multiple of
 * n_rhs, input beyond the limit, memory not on the current device), WD_ECUDA.  wd_action_static_error() returns the
 * text for the calling thread's last failure of this call ("" after a success); it never returns NULL. */
#define WD_STATIC_MAX_ROWS 33554432        /* 2^25 = 16384 thread blocks x 2048 rows */
#define WD_STATIC_SCRATCH_BYTES 2097408    /* 16384 x WD_MAX_RHS doubles + one 256-byte line for the counter */
int wd_action_static(int n_rhs, size_t n_complex, const double* X_native_dev, double* S_dev, void* cuda_stream);
const char* wd_action_static_error(void);

/* Per-class device timing for measurement (bench.py's roofline line).  wd_profile(ctx, 1) makes every
 * later hop / BLAS1 / force launch record a CUDA event pair on the context's stream (a few
 * microseconds of host time each; leave it off when timing whole calls).  wd_profile_read
 * synchronises the stream, adds up the event-pair durations recorded since the previous read into
 * ms[class] (milliseconds) and count[class] (launch groups), class = WD_PROF_*, both arrays of
 * WD_PROF_N, and resets the record.  Errors: WD_EINVAL (null), WD_ECUDA. */
enum { WD_PROF_HOP32 = 0, WD_PROF_HOP64 = 1, WD_PROF_BLAS = 2, WD_PROF_FORCE = 3, WD_PROF_LAYOUT = 4, WD_PROF_N = 5 };
int wd_profile(wd_ctx* ctx, int enable);
int wd_profile_read(wd_ctx* ctx, double* ms_host, long long* count_host);

/* Residual history: what the paper plots in Fig. 1-5, |D x - b| / |b| against the iteration number,
 * one curve per pseudo-fermion.  hist_dev is the caller's DEVICE buffer of capacity rows of WD_MAX_RHS doubles (NULL or
 * capacity 0 switches the record off; it is off by default and costs nothing then).  While it is set, every
 * wd_solve_block (and the calls built on it) writes row k, column i = the estimate of |phi_i - A x_i| / |phi_i| after
 * its k-th low-precision BiCGStab iteration, k counted from 0 over the whole solve (across the restarts of the outer
 * loop), for k < capacity; info.inner_iters_total rows are valid after the call.  The estimate is the RECURSIVE residual of
 * the fp32 (or 16-bit) even/odd system scaled back to the fp64 one, i.e. what the iteration itself sees; the true
 * residual at the end is info.relres.  A column that has converged keeps its last value.  Routes: the default solver and
 * WD_SOLVER_RELIABLE_H16 (for WD_SOLVER_GL_FLEX the rows are the preconditioner's inner iterations; the fp64 blocked
 * solvers write nothing).  The buffer must stay valid while it is set.  Errors: WD_EINVAL. */
int wd_set_residual_history(wd_ctx* ctx, double* hist_dev, int capacity);

/* What the fp32 inner solver of wd_solve_block will run for (n_rhs, recon) with the options as they are
 * now, so that a measurement can count the right bytes without repeating the library's dispatch rules: plan_host is
 * an array of WD_PLAN_N ints, [WD_PLAN_HOP_KERNEL] = the kernel that serves the four hop launches of an iteration
 * (WD_HOP_KERNEL_*), [WD_PLAN_MERGED] = 1 for the merged x,r,p update schedule (WD_OPT_MERGE: 23 vector passes per
 * iteration, seven-sum epilogue in the second hop pair), 0 for the textbook order (25), [WD_PLAN_PAIRED] = 1 for the
 * x-paired form, [WD_PLAN_KERNELS_PER_ITER] = kernel launches per BiCGStab iteration (6 or 7).  Host only, launches
 * nothing.  Errors: WD_EINVAL (null, n_rhs out of range, bad recon). */
enum { WD_HOP_KERNEL_REGISTER = 0, WD_HOP_KERNEL_RING = 1, WD_HOP_KERNEL_ZMARCH = 2 };
enum { WD_PLAN_HOP_KERNEL = 0, WD_PLAN_MERGED = 1, WD_PLAN_PAIRED = 2, WD_PLAN_KERNELS_PER_ITER = 3, WD_PLAN_N = 4 };
int wd_inner_plan(const wd_ctx* ctx, int n_rhs, int recon, int* plan_host);

/* Number of kernel launches this context has enqueued since creation (for bench.py's count). */
long long wd_launch_count(const wd_ctx* ctx);

const char* wd_strerror(int code);
const char* wd_last_error(const wd_ctx* ctx);
const char* wd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WD_H */
