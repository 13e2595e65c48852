"""ugks_residual_noalloc (include/ugks.h): the residual entry point for callers that cannot allocate device memory.

Some users of libugks only want the O11 residual of two W fields and have no way to get scratch memory for it: a
convergence monitor or logging hook running inside a process whose device memory was handed to a pool up front (cudaMalloc
fails there and the hook has no handle to the pool), or a time loop that cannot take the device-wide synchronisation of
cudaMalloc / cudaFree.  For them the per-block partial sums live in a fixed 512 KiB array inside libugks.so instead of the
caller's workspace, which caps the field at UGKS_NOALLOC_MAX_CELLS cells and makes every call on a device share that array.

This file is collected last on purpose (pytest -x stops at the first failure): the existing path, ugks_residual of a context,
is the reference, and the new entry point must agree with it within the residual tolerance the parity tests use (RES_RTOL),
on calls in a row that leave different amounts of stale data in the shared array.
"""
import ctypes as C

import numpy as np
import pytest

import workloads

RES_RTOL = 1e-10                       # tests/test_gpu_parity.py compares residuals at this relative tolerance


@pytest.fixture(scope="module", autouse=True)
def _built_library():
    from paper_1810_08137_b200 import build
    build.build()


def test_sizes_beyond_the_static_array_are_refused():
    """The size check comes before any CUDA call, so it can run without a GPU; nothing is launched and the message names the limit."""
    from paper_1810_08137_b200 import binding
    L = binding.lib()
    buf = C.create_string_buffer(320)
    p = C.c_void_p(256)                                                       # never dereferenced on these paths
    assert L.ugks_residual_noalloc(p, p, binding.NOALLOC_MAX_CELLS + 1, p, None, buf, len(buf)) == 1
    assert b"UGKS_NOALLOC_MAX_CELLS = 1048576" in buf.value
    assert L.ugks_residual_noalloc(p, p, 0, p, None, buf, len(buf)) == 1 and b"ncells" in buf.value
    assert L.ugks_residual_noalloc(None, p, 8, p, None, buf, len(buf)) == 1 and b"NULL" in buf.value
    assert L.ugks_residual_noalloc(p, p, 1 << 40, p, None, None, 0) == 1      # the message buffer is optional


def _context_residuals(p, steps):
    """The existing path: step a context and collect (W^n, W^{n+1}, ugks_residual) of every step."""
    import torch
    from paper_1810_08137_b200 import Ugks
    W, f, _ = workloads.initial_state(p)
    g = Ugks(p)
    g.set_state(W, f)
    out = []
    Wn = g.W(torch.empty((p.J, p.I, 4), dtype=torch.float64, device="cuda"))
    for _ in range(steps):
        g.step(1)
        Wp = g.W(torch.empty((p.J, p.I, 4), dtype=torch.float64, device="cuda"))
        out.append((Wn, Wp, g.residual()))
        Wn = Wp
    g.close()
    return out


@pytest.mark.gpu
def test_matches_the_context_residual_on_calls_in_a_row():
    import torch
    from paper_1810_08137_b200 import residual_noalloc
    big = _context_residuals(workloads.channel_config("C2", I=131, J=37), 2)          # 4847 cells: 38 blocks, ragged last block
    small = _context_residuals(workloads.channel_config("C1"), 2)                     # 512 cells: 4 blocks
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    # big, big, small, small, big: the small calls find the big call's partials beyond their own 4 blocks, and the last big
    # call finds the small call's in its first 4; none of that may leak into a result
    for Wn, Wp, ref in (big[0], big[1], small[0], small[1], big[0]):
        assert np.all(ref > 0.0)
        res = residual_noalloc(Wn, Wp, out=out).cpu().numpy()                         # .cpu() synchronises the stream
        assert np.all(np.abs(res - ref) <= RES_RTOL * np.abs(ref)), (res, ref)
    # identical fields: zero residual, not whatever the previous call left behind
    res = residual_noalloc(big[0][1], big[0][1], out=out).cpu().numpy()
    assert np.all(res == 0.0), res
    # a device result tensor made by the binding (torch), and a non-default stream
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        r2 = residual_noalloc(small[1][0], small[1][1])
    s.synchronize()
    assert np.all(np.abs(r2.cpu().numpy() - small[1][2]) <= RES_RTOL * np.abs(small[1][2]))
