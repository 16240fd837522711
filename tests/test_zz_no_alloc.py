"""mspcg_dot2_noalloc (include/mspcg.h): the inner products of eq. 18 with the scratch in the library's static device array,
for callers that cannot allocate.  Checked against the EXISTING path -- k_dot2 with its scratch scalars in the caller's
workspace, reached through mspcg_residual (|b - D^dag D 0| = |b|) -- at the
fp64 tolerance of the other tests (1e-12), on two calls in a row that share the array.  Collected last on purpose
(the suite runs with pytest -x).  Needs no state from other tests: it builds its own context."""
import ctypes as C

import numpy as np
import pytest

from paper_2104_05615_b200 import F64, Mspcg, dot2_noalloc, load_library, synth

pytestmark = pytest.mark.gpu

TOL = 1e-12


def test_dot2_noalloc_matches_workspace_path_on_two_calls_in_a_row():
    import torch
    lib = load_library()
    dims, Ls, block = (4, 4, 6, 8), 8, (2, 2, 6, 4)
    g = Mspcg(dims, Ls, 1.5, 0.5, 1.8, 0.02, block)
    g.configure(F64, F64, 18)
    g.load_gauge(synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 11), dims), -1)
    b1 = torch.as_tensor(synth.gaussian_spinor_abi(dims, Ls, 1).reshape(-1)).cuda()       # 73728 reals: 4.5 chunks, ragged tail
    b2 = torch.as_tensor(synth.gaussian_spinor_abi(dims, Ls, 2).reshape(-1)).cuda() * 3.0
    zero = torch.zeros_like(b1)
    # existing path: |b - A 0| through k_dot2 into the workspace scalars
    n1 = g.residual(b1, zero)[1]
    n2 = g.residual(b2, zero)[1]
    short = b2[: 16384 + 5].contiguous()                                                  # fewer chunks than the call before: stale partial sums stay behind
    out = torch.full((3, 2), -7.0, dtype=torch.float64, device="cuda")
    dot2_noalloc(b1, b1, None, out[0])                                                    # warm-up: the first call on a device looks up the symbol's address
    out.fill_(-7.0)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    dot2_noalloc(b1, b1, b2, out[0])                                                      # call 1
    dot2_noalloc(b2, b2, b1, out[1])                                                      # call 2, same stream, straight after
    dot2_noalloc(short, short, None, out[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                                          # nothing was allocated on the device
    o = out.cpu().numpy()
    assert abs(np.sqrt(o[0, 0]) - n1) <= TOL * n1, (np.sqrt(o[0, 0]), n1)
    assert abs(np.sqrt(o[1, 0]) - n2) <= TOL * n2, (np.sqrt(o[1, 0]), n2)
    # <b1, b2>: by polarisation from three norms of the existing path, and directly
    n12 = g.residual(b1 + b2, zero)[1]
    cross = 0.5 * (n12 ** 2 - n1 ** 2 - n2 ** 2)
    assert abs(o[0, 1] - cross) <= 1e-11 * n1 * n2
    assert o[0, 1] == o[1, 1]                                                             # same products, same fixed summation order
    assert abs(o[0, 1] - float(torch.dot(b1, b2))) <= TOL * n1 * n2
    assert abs(o[2, 0] - float(torch.dot(short, short))) <= TOL * o[2, 0] and o[2, 1] == 0.0
    # bitwise reproducible from call to call (fixed order, no atomics on the sums)
    again = torch.empty(2, dtype=torch.float64, device="cuda")
    dot2_noalloc(b1, b1, b2, again)
    assert np.array_equal(again.cpu().numpy(), o[0])
    # empty input, and the size limit
    dot2_noalloc(b1[:0], b1[:0], None, again)
    assert not again.cpu().numpy().any()
    nmax = lib.mspcg_dot2_noalloc_max_reals()
    assert nmax == 1 << 29
    rc = lib.mspcg_dot2_noalloc(C.c_void_p(b1.data_ptr()), C.c_void_p(b1.data_ptr()), None, nmax + 1, C.c_void_p(again.data_ptr()), None)
    assert rc == -1 and b"outside" in lib.mspcg_noalloc_last_error()
    rc = lib.mspcg_dot2_noalloc(None, C.c_void_p(b1.data_ptr()), None, 16, C.c_void_p(again.data_ptr()), None)
    assert rc == -1 and b"null" in lib.mspcg_noalloc_last_error()
    g.close()
