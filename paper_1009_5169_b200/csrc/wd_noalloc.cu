// wd_noalloc.cu -- wd_action_static: the per-column action S_i = |x_i|^2 (eq. 2.2; the quantity the
// Metropolis step of PAPER.md:60 compares) for callers that cannot allocate device memory.
//
// Who that is.  wd_action needs a context, and a context needs a workspace the caller cudaMalloc's and hands over
// (gigabytes at 24^4, because it also holds the solver's vectors).  Two kinds of caller cannot do that: a lattice code
// that has already given every byte of the card to its own field arena (there is nothing left to ask the driver for,
// and going through the driver would bypass the arena's accounting), and code that runs while other streams are busy
// and must not stall them -- cudaMalloc and cudaFree synchronise the whole device.  Such a caller holds a native fp64
// block in memory of its own and only wants its norm per column.
//
// What the kernel needs besides its input and output is one partial sum per (thread block, column) and a ticket
// counter that tells the last block to add the partials up.  Here that scratch is a file-scope __device__ array of fixed
// size: it is part of the library image, every GPU that loads libwd.so carries it (WD_STATIC_SCRATCH_BYTES, about
// 2 MiB) until the process exits, and nothing is allocated or freed by the call -- no cudaMalloc, no cudaFree, no
// pinned host buffer, no context.  The fixed size is what bounds the input: see WD_STATIC_MAX_ROWS in include/wd.h.
//
// Summation order.  Block b adds rows [b * SEG_ROWS, (b+1) * SEG_ROWS) (a row = the n_rhs complex numbers that share
// one flat index / n_rhs), and the last block adds the per-block partials in index order.  The order therefore depends
// only on (n_rhs, n_complex), not on the SM count or on block scheduling: the same input gives the same bits on any GPU.
// Everything is fp64.  This file shares no code with the context path (csrc/wd_md.cu action_kernel).
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/wd.h"

namespace {

constexpr int SEG_ROWS = 2048;                                   // rows one thread block adds up
constexpr unsigned MAX_BLOCKS = (unsigned)(WD_STATIC_MAX_ROWS / SEG_ROWS);
constexpr size_t PARTIAL_DOUBLES = (size_t)MAX_BLOCKS * WD_MAX_RHS;
constexpr int MAX_DEVICES = 64;

static_assert(WD_STATIC_MAX_ROWS % SEG_ROWS == 0, "the row limit is a whole number of block segments");
static_assert(PARTIAL_DOUBLES * sizeof(double) + 256 == WD_STATIC_SCRATCH_BYTES, "wd.h states the size of the static scratch");

// The scratch itself: [column][block] partial sums, then (in a 256-byte line of its own) the ticket counter.
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and must never be
// passed to a kernel as a pointer; scratch_for_current_device() below turns it into one.
struct StaticScratch {
    double partials[PARTIAL_DOUBLES];
    unsigned int ticket;
    unsigned int pad[63];
};
static __device__ __align__(256) StaticScratch g_static_scratch;

thread_local const char* t_err = "";

int fail(int code, const char* msg) {
    t_err = msg;
    return code;
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device (each device that loads the
// library has its own copy of the array at its own address).
std::mutex g_mu;
StaticScratch* g_scratch_ptr[MAX_DEVICES] = {};

cudaError_t scratch_for_current_device(int dev, StaticScratch** out) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        StaticScratch* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

// Threads of a block: a multiple of 32 and of n with at least n warps (thread t always works on column t % n, and
// warp w < n adds up column w).  n = 1..16 gives 256..512 threads.
int block_threads(int n) { return 32 * n * ((8 + n - 1) / n); }

__global__ void __launch_bounds__(512)
action_static_kernel(long rows, int n, const double2* __restrict__ X, StaticScratch* __restrict__ scr, double* __restrict__ S) {
    __shared__ double sh[512];
    __shared__ bool is_last;
    const int B = blockDim.x, t = threadIdx.x;
    const int per = B / n;            // threads per column
    const int r = t % n, q = t / n;   // my column, my index among its threads
    const int warp = t >> 5, lane = t & 31, nwarps = B >> 5;
    const unsigned grid = gridDim.x;

    // this block's segment: element index = row * n + column, and B is a multiple of n, so t + k * B stays in column r
    const long row0 = (long)blockIdx.x * SEG_ROWS;
    const long row1 = row0 + SEG_ROWS < rows ? row0 + SEG_ROWS : rows;
    const long e1 = row1 * n;
    double s = 0.0;
    for (long i = row0 * n + t; i < e1; i += B) {
        const double2 a = X[i];
        s += a.x * a.x + a.y * a.y;
    }
    sh[r * per + q] = s;
    __syncthreads();
    if (warp < n) {
        double w = 0.0;
        for (int j = lane; j < per; j += 32) w += sh[warp * per + j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
        if (lane == 0) scr->partials[(size_t)warp * grid + blockIdx.x] = w;
    }
    __threadfence();
    __syncthreads();
    if (t == 0) is_last = (atomicAdd(&scr->ticket, 1u) == grid - 1);
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // last block to finish: column by column, every thread adds a strided slice of the partials, then warps, then one thread
    for (int col = 0; col < n; ++col) {
        const double* p = scr->partials + (size_t)col * grid;
        double w = 0.0;
        for (unsigned g = t; g < grid; g += B) w += __ldcg(p + g);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
        if (lane == 0) sh[col * 32 + warp] = w;   // nwarps <= 16 < 32
    }
    __syncthreads();
    if (t < n) {
        double w = 0.0;
        for (int k = 0; k < nwarps; ++k) w += sh[t * 32 + k];
        S[t] = w;
    }
    if (t == 0) scr->ticket = 0u;   // leave the counter ready for the next call (the host also clears it before each launch)
}

}  // namespace

extern "C" {

const char* wd_action_static_error(void) { return t_err; }

int wd_action_static(int n_rhs, size_t n_complex, const double* X_native_dev, double* S_dev, void* cuda_stream) {
    t_err = "";
    if (n_rhs < 1 || n_rhs > WD_MAX_RHS) return fail(WD_EINVAL, "wd_action_static: n_rhs must be 1..WD_MAX_RHS");
    if (!X_native_dev || !S_dev) return fail(WD_EINVAL, "wd_action_static: null pointer");
    if (((size_t)X_native_dev & 15) != 0 || ((size_t)S_dev & 7) != 0)
        return fail(WD_EINVAL, "wd_action_static: X must be 16-byte aligned and S 8-byte aligned");
    if (n_complex == 0 || n_complex % (size_t)n_rhs != 0)
        return fail(WD_EINVAL, "wd_action_static: n_complex must be a positive multiple of n_rhs");
    const size_t rows = n_complex / (size_t)n_rhs;
    if (rows > (size_t)WD_STATIC_MAX_ROWS)
        return fail(WD_EINVAL, "wd_action_static: input too large for the static scratch: n_complex / n_rhs exceeds "
                               "WD_STATIC_MAX_ROWS (use wd_action with a context and workspace instead)");

    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(WD_ECUDA, "wd_action_static: cudaGetDevice failed (no CUDA device?)");
    if (dev < 0 || dev >= MAX_DEVICES) return fail(WD_EINVAL, "wd_action_static: device ordinal out of range");
    // the scratch used is the current device's copy, so X and S have to live there too
    cudaPointerAttributes ax, ao;
    if (cudaPointerGetAttributes(&ax, X_native_dev) != cudaSuccess || cudaPointerGetAttributes(&ao, S_dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(WD_ECUDA, "wd_action_static: cudaPointerGetAttributes failed");
    }
    const bool x_ok = (ax.type == cudaMemoryTypeDevice && ax.device == dev) || ax.type == cudaMemoryTypeManaged;
    const bool s_ok = (ao.type == cudaMemoryTypeDevice && ao.device == dev) || ao.type == cudaMemoryTypeManaged;
    if (!x_ok || !s_ok) return fail(WD_EINVAL, "wd_action_static: X and S must be device memory of the current device");

    StaticScratch* scr = nullptr;
    if (scratch_for_current_device(dev, &scr) != cudaSuccess || !scr) {
        cudaGetLastError();
        return fail(WD_ECUDA, "wd_action_static: cudaGetSymbolAddress of the static scratch failed");
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the only part of the scratch that has to start at zero; the partials are overwritten before they are read
    if (cudaMemsetAsync(&scr->ticket, 0, sizeof(unsigned int), st) != cudaSuccess) {
        cudaGetLastError();
        return fail(WD_ECUDA, "wd_action_static: clearing the ticket counter failed");
    }
    const unsigned grid = (unsigned)((rows + SEG_ROWS - 1) / SEG_ROWS);   // <= MAX_BLOCKS by the check above
    action_static_kernel<<<grid, block_threads(n_rhs), 0, st>>>((long)rows, n_rhs, (const double2*)X_native_dev, scr, S_dev);
    if (cudaGetLastError() != cudaSuccess) return fail(WD_ECUDA, "wd_action_static: kernel launch failed");
    return WD_OK;
}

}  // extern "C"
