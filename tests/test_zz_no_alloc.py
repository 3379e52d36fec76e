"""lqcd_coarse_mult_half_noalloc_f32: the coarse operator on half storage with its scratch in a file-scope
`static __device__` array of the library (LQCD_NOALLOC_SCRATCH_BYTES = 16 MiB) instead of a caller-owned workspace --
for callers that cannot call cudaMalloc (CUDA graph capture, serving loops).  include/lqcd_b200.h states the limit and
the sharing rule.

Checked here against the EXISTING path (lqcd_coarse_mult_half_f32 with a workspace) on calls made back to back, so
that the second call runs on whatever the first one left in the shared array, and against the oracle's nine-block
operator (Eq. 4 with the blocks of Eq. 7) for one problem.  This file is collected last on purpose
(the suite runs with pytest -x): it must pass alone in a fresh process and after every other test.
"""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle
from problems import expand_half, rel_l2

pytestmark = pytest.mark.gpu
TOL_F32 = 2e-6  # the single-application fp32 bar of tests/test_gpu_half.py


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available()
    import paper_2111_05012_b200 as lq
    return lq


def random_half_problem(seed, cdims, nvec):
    rng = np.random.default_rng(seed)
    vc, n = int(np.prod(cdims)), 2 * nvec
    Ah = 0.1 * (rng.standard_normal((vc, 5, n, n)) + 1j * rng.standard_normal((vc, 5, n, n)))
    Ah[:, 0] += np.eye(n)  # the recipe of tests/test_gpu_half.py::test_half_storage_edge_sizes
    x = li.coarse_vector(rng, vc, nvec)
    return np.ascontiguousarray(Ah.astype(np.complex64)), np.ascontiguousarray(x.astype(np.complex64))


def both_paths(lq, Ah, x, cdims, nvec, dagger):
    import torch
    A, xd = torch.from_numpy(Ah).cuda(), torch.from_numpy(x).cuda()
    y_ws = torch.full_like(xd, 7.0)
    lq.coarse_mult_half(y_ws, xd, A, cdims, nvec, dagger=dagger)         # existing path, caller-owned workspace
    y_na = torch.full_like(xd, -3.0)                                     # every entry must be overwritten
    lq.coarse_mult_half_noalloc(y_na, xd, A, cdims, nvec, dagger=dagger)  # static scratch
    torch.cuda.synchronize()
    return y_ws, y_na


def test_two_calls_in_a_row_match_the_workspace_path(lq):
    """Call 1 on a larger lattice fills the shared array; call 2 on a smaller lattice with another row length, and
    call 3 on the first shape again with new data, run on those left-overs.  Each must match the workspace path
    (same kernels: the same bits) and, for the problems the oracle finishes quickly, the oracle."""
    import torch
    calls = [((6, 4, 4, 2), 32, False, 11), ((3, 2, 5, 2), 3, True, 12), ((6, 4, 4, 2), 32, True, 13),
             ((2, 4, 2, 2), 20, False, 14)]
    for cdims, nvec, dagger, seed in calls:
        Ah, x = random_half_problem(seed, cdims, nvec)
        y_ws, y_na = both_paths(lq, Ah, x, cdims, nvec, dagger)
        assert rel_l2(y_na.cpu().numpy(), y_ws.cpu().numpy()) <= TOL_F32, (cdims, nvec, dagger)
        assert torch.equal(y_na, y_ws), (cdims, nvec, dagger)
        ref = oracle.coarse_mult(x, expand_half(Ah, cdims, nvec), cdims, dagger=dagger)
        assert rel_l2(y_na.cpu().numpy(), ref) <= TOL_F32, (cdims, nvec, dagger)


def test_same_problem_twice_gives_the_same_bits(lq):
    import torch
    cdims, nvec = (4, 2, 2, 3), 8
    Ah, x = random_half_problem(21, cdims, nvec)
    A, xd = torch.from_numpy(Ah).cuda(), torch.from_numpy(x).cuda()
    y1, y2 = torch.empty_like(xd), torch.empty_like(xd)
    lq.coarse_mult_half_noalloc(y1, xd, A, cdims, nvec)
    lq.coarse_mult_half_noalloc(y2, xd, A, cdims, nvec)
    torch.cuda.synchronize()
    assert torch.equal(y1, y2)


def test_largest_problem_that_fits_and_no_device_memory_is_taken(lq):
    """Config 4's coarse lattice (8^3 x 16, nvec 32) needs exactly LQCD_NOALLOC_SCRATCH_BYTES.  Synthetic blocks made
    on the device (the oracle is not needed: the comparison is with the workspace path).  cudaMemGetInfo before and
    after the calls: the entry point must not take device memory."""
    import torch
    cdims, nvec = (8, 8, 8, 16), 32
    assert lq.lib().lqcd_coarse_half_workspace_bytes(lq._i4(cdims), nvec, 4) == lq.NOALLOC_SCRATCH_BYTES
    vc, n = 8 * 8 * 8 * 16, 64
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    A = torch.view_as_complex(torch.randn((vc, 5, n, n, 2), generator=g, device="cuda", dtype=torch.float32) * 0.05)
    x = torch.view_as_complex(torch.randn((vc, 2, nvec, 2), generator=g, device="cuda", dtype=torch.float32))
    ws = lq.coarse_half_workspace(cdims, nvec)
    y_ws, y_na = torch.empty_like(x), torch.empty_like(x)
    lq.coarse_mult_half(y_ws, x, A, cdims, nvec, ws=ws)
    lq.coarse_mult_half_noalloc(y_na, x, A, cdims, nvec)  # first call on this device may resolve the symbol address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        lq.coarse_mult_half_noalloc(y_na, x, A, cdims, nvec)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
    assert torch.equal(y_na, y_ws)
    assert rel_l2(y_na.cpu().numpy(), y_ws.cpu().numpy()) <= TOL_F32


def test_a_problem_beyond_the_static_scratch_is_refused(lq):
    """One coarse site more in t than fits: LQCD_EUNSUPPORTED, a message with both sizes, nothing launched (the size
    check comes before any pointer is looked at, so small stand-in buffers do)."""
    import torch
    buf = torch.zeros(64, device="cuda", dtype=torch.float32)
    out = torch.zeros(64, device="cuda", dtype=torch.float32)
    n0 = lq.lib().lqcd_launch_count()
    for cdims, nvec in (((8, 8, 8, 17), 32), ((16, 16, 16, 9), 8)):
        rc = lq.lib().lqcd_coarse_mult_half_noalloc_f32(lq._dev_ptr(out), lq._dev_ptr(buf), lq._dev_ptr(buf),
                                                        lq._i4(cdims), nvec, 0, None)
        assert rc == lq.EUNSUPPORTED
        msg = lq.lib().lqcd_last_error().decode()
        assert "LQCD_NOALLOC_SCRATCH_BYTES" in msg and str(lq.NOALLOC_SCRATCH_BYTES) in msg, msg
    assert lq.lib().lqcd_launch_count() == n0
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
    # the binding raises the same refusal
    with pytest.raises(lq.LqcdError):
        vc = 16 * 16 * 16 * 9
        x = torch.zeros((vc, 2, 8), device="cuda", dtype=torch.complex64)
        A = torch.zeros((vc, 5, 16, 16), device="cuda", dtype=torch.complex64)
        lq.coarse_mult_half_noalloc(torch.empty_like(x), x, A, (16, 16, 16, 9), 8)
