"""wd_action_static: the per-column action |x_i|^2 for callers that cannot allocate device memory.

Some users of libwd.so cannot call cudaMalloc: a lattice code that has handed the whole card to its own field arena,
or code that must not stall its other streams (cudaMalloc / cudaFree synchronise the device).  wd_action is closed to
them because a context needs a caller-allocated workspace.  wd_action_static takes only the input block, an output
array and a stream; its scratch (per-block partial sums, a ticket counter) is a fixed array inside the library, which
is why the input size is bounded (WD_STATIC_MAX_ROWS) and why every call reuses what the previous call left behind.

The GPU test makes two calls in a row, on different blocks and column counts, so that a call which trusted leftover
scratch from the one before it would give a wrong sum; each result is compared with wd_action (the context path) at the
rtol = 1e-13 that tests/test_gpu_parity.py::test_refresh_and_action uses for the action, and with the oracle.  The file
name sorts after the other test files on purpose: pytest -x stops at the first failure, and a failure here should not
hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

import wd_inputs as wi


def _wd():
    import paper_1009_5169_b200 as pkg
    return pkg


def test_static_entry_rejects_what_it_cannot_serve_before_touching_the_gpu():
    """Argument checks come before any CUDA call, so they can be exercised without a device: sizes beyond the static
    scratch, column counts outside 1..16, null and misaligned pointers, a length that is not whole rows."""
    pkg = _wd()
    L = pkg.wd.lib()
    fake = ctypes.c_void_p(1 << 20)   # aligned, never dereferenced: every case below fails a check first
    n = 5
    too_big = (pkg.wd.STATIC_MAX_ROWS + 1) * n
    assert L.wd_action_static(n, too_big, fake, fake, None) == pkg.wd.EINVAL
    msg = L.wd_action_static_error().decode()
    assert "too large" in msg and "WD_STATIC_MAX_ROWS" in msg, msg
    assert L.wd_action_static(0, 10, fake, fake, None) == pkg.wd.EINVAL
    assert L.wd_action_static(pkg.wd.MAX_RHS + 1, 17, fake, fake, None) == pkg.wd.EINVAL
    assert L.wd_action_static(n, 10, None, fake, None) == pkg.wd.EINVAL
    assert L.wd_action_static(n, 10, fake, None, None) == pkg.wd.EINVAL
    assert L.wd_action_static(n, 10, ctypes.c_void_p((1 << 20) + 8), fake, None) == pkg.wd.EINVAL
    assert L.wd_action_static(n, 11, fake, fake, None) == pkg.wd.EINVAL     # not a multiple of n_rhs
    assert L.wd_action_static(n, 0, fake, fake, None) == pkg.wd.EINVAL
    assert L.wd_action_static_error().decode() != ""
    # the limits the header states are the ones the binding carries
    hdr = open(pkg.wd.HERE + "/../include/wd.h").read()
    assert f"#define WD_STATIC_MAX_ROWS {pkg.wd.STATIC_MAX_ROWS}" in hdr
    assert f"#define WD_STATIC_SCRATCH_BYTES {pkg.wd.STATIC_SCRATCH_BYTES}" in hdr


@pytest.mark.gpu
def test_static_action_matches_the_context_path_on_two_calls_in_a_row():
    pkg = _wd()
    from oracle import wd_oracle as orc
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731

    # two different blocks: 8^3 x 16 with 5 columns (98304 rows = 48 whole segments of the static kernel) and
    # 6 x 6 x 6 x 10 with 3 columns (25920 rows: 13 segments, the last one short; 6.3 segments per parity half)
    cases = [((8, 8, 8, 16), wi.BC_SF, 5, 21), ((6, 6, 6, 10), wi.BC_PERIODIC, 3, 22)]
    blocks = []
    for dims, bc, n, seed in cases:
        eta = wi.spinor_field(dims, n, seed, bc)
        ctx = pkg.Context(dims, 0.13, bc=bc, max_rhs=n)
        E = ctx.pack(dev(eta))
        want = {sel: np.array(ctx.action(E, n, sel)) for sel in (pkg.PARITY_BOTH, pkg.PARITY_EVEN, pkg.PARITY_ODD)}
        blocks.append((dims, n, eta, E, want))
        ctx.close()          # the static entry point needs no context: none is alive from here on
    torch.cuda.synchronize()

    # the caller's output arrays exist before the calls; the calls themselves must not allocate
    outs = [torch.full((n,), -1.0, dtype=torch.float64, device="cuda") for _, n, _, _, _ in blocks]
    # set-up call, as include/wd.h asks for: the first call on a device looks up the scratch array's address, and the
    # driver may load the library's kernels (and the array itself) only then
    pkg.action_static(blocks[1][3], blocks[1][1], out=outs[1])
    torch.cuda.synchronize()
    outs[1].fill_(-1.0)
    free_before = torch.cuda.mem_get_info()[0]
    # call 1 and call 2 back to back on one stream, no synchronisation in between
    for (dims, n, eta, E, want), out in zip(blocks, outs):
        pkg.action_static(E, n, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before      # the driver handed out no device memory
    for (dims, n, eta, E, want), out in zip(blocks, outs):
        got = out.cpu().numpy()
        assert np.allclose(got, want[pkg.PARITY_BOTH], rtol=1e-13, atol=0.0), (got, want[pkg.PARITY_BOTH])
        assert np.allclose(got, orc.action(eta), rtol=1e-13, atol=0.0)

    # and again in the other order, one parity half each: the scratch now holds the leftovers of a larger call
    for (dims, n, eta, E, want), out in reversed(list(zip(blocks, outs))):
        for sel in (pkg.PARITY_ODD, pkg.PARITY_EVEN):
            got = pkg.action_static(E, n, sel, out=out).cpu().numpy()
            assert np.allclose(got, want[sel], rtol=1e-13, atol=0.0), (sel, got, want[sel])
    # same input, same bits: the summation order is fixed by the sizes alone
    a = pkg.action_static(blocks[0][3], blocks[0][1]).cpu().numpy()
    b = pkg.action_static(blocks[0][3], blocks[0][1]).cpu().numpy()
    assert np.array_equal(a, b)


@pytest.mark.gpu
def test_static_action_rejects_memory_that_is_not_on_the_device():
    pkg = _wd()
    L = pkg.wd.lib()
    host = torch.zeros(64, dtype=torch.float64)
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    rc = L.wd_action_static(4, 32, ctypes.c_void_p(host.data_ptr()), ctypes.c_void_p(out.data_ptr()), None)
    assert rc == pkg.wd.EINVAL, rc
    assert "device memory" in L.wd_action_static_error().decode()
