"""dmrg_gemv_trans_static (include/dmrg_b200.h): gemv_trans (Alg. 3 lines 3 / 12; Alg. 4) for callers that may not
allocate -- no plan, no cudaMalloc; the kernel's cross-CTA scratch is a file-scope device array shared by all calls.

Collected LAST on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide another test.
Checked: the new entry point against the existing path (dmrg_gemv_trans of a plan) and against numpy, on two calls in a row
that reuse the scratch (different basis sizes and vectors, so stale partial sums or a stale counter would show), for an unaligned
vector (scalar path), for a size that fills all 1024 scratch rows, that the device allocator is untouched, and the size limits."""
import ctypes as C

import numpy as np
import pytest

from dmrg_inputs import random_vector, make_config
from gpu_common import to_dev

pytestmark = pytest.mark.gpu

TOL = 4e-12        # x sqrt(n): the tolerance of test_blas2_kernels_match_numpy for the existing path


@pytest.fixture(scope="module")
def lib():
    import torch
    assert torch.cuda.is_available()
    import paper_1309_5571_b200 as lib
    lib.load_library()
    return lib


def test_static_gemv_trans_matches_existing_path_two_calls_in_a_row(lib):
    import torch
    p = make_config("cfg2", 160)
    plan = lib.Plan(p, k_max=32)
    n = plan.n
    ldv = n + 1                                             # odd stride: the columns are not all 16-byte aligned -> scalar path
    Vh = np.stack([random_vector(ldv, 9100 + j) for j in range(32)])
    V = to_dev(Vh)
    out = torch.full((32,), float("nan"), dtype=torch.float64, device="cuda")
    w1, w2 = random_vector(n, 9201), random_vector(n, 9202)
    # two calls in a row on the same stream, second one with fewer columns and another vector: it must not see the first one's sums
    for k, wh in ((32, w1), (5, w2), (17, w1)):
        w = to_dev(wh)
        ref = plan.gemv_trans(V, k, w).clone()
        got = lib.gemv_trans_static(V, k, w, out, n=n)[:k].clone()
        torch.cuda.synchronize()
        assert float((got - ref).abs().max()) <= TOL * np.sqrt(n)
        assert np.max(np.abs(got.cpu().numpy() - Vh[:k, :n] @ wh)) <= TOL * np.sqrt(n)
    # even stride and aligned pointers: the 16-byte path; back to back without a synchronisation in between
    V2 = to_dev(np.ascontiguousarray(Vh[:, :n + (n % 2)]))
    n2 = n - (n % 2)
    oa = torch.empty(32, dtype=torch.float64, device="cuda"); ob = torch.empty(32, dtype=torch.float64, device="cuda")
    wa, wb = to_dev(w1[:n2].copy()), to_dev(w2[:n2].copy())
    lib.gemv_trans_static(V2, 24, wa, oa, n=n2)
    lib.gemv_trans_static(V2, 24, wb, ob, n=n2)
    torch.cuda.synchronize()
    assert np.max(np.abs(oa[:24].cpu().numpy() - Vh[:24, :n2] @ w1[:n2])) <= TOL * np.sqrt(n)
    assert np.max(np.abs(ob[:24].cpu().numpy() - Vh[:24, :n2] @ w2[:n2])) <= TOL * np.sqrt(n)
    # bitwise reproducible (fixed-order reduction), like the existing path
    oc = torch.empty(32, dtype=torch.float64, device="cuda")
    lib.gemv_trans_static(V2, 24, wb, oc, n=n2)
    torch.cuda.synchronize()
    assert torch.equal(ob[:24], oc[:24])
    plan.close()


def test_static_gemv_trans_full_grid_and_no_device_allocation(lib):
    """n large enough for the grid to reach the 1024 rows of the scratch; the driver's free-memory figure does not move across
    the calls (no cudaMalloc / cudaFree on the way) and neither does torch's allocator."""
    import torch
    n, k = 1_500_001, 8
    rng = np.random.default_rng(77)
    Vh = rng.standard_normal((k, n)); wh = rng.standard_normal(n)
    V, w = to_dev(Vh), to_dev(wh)
    out = torch.empty(k, dtype=torch.float64, device="cuda")
    lib.gemv_trans_static(V, k, w, out)                      # first call on this device: symbol address looked up here
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    a0 = torch.cuda.memory_allocated()
    for _ in range(2):
        lib.gemv_trans_static(V, k, w, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_allocated() == a0
    assert np.max(np.abs(out.cpu().numpy() - Vh @ wh)) <= TOL * np.sqrt(n)


def test_static_gemv_trans_rejects_sizes_beyond_the_maximum(lib):
    import torch
    L = lib.load_library()
    V = torch.zeros((34, 64), dtype=torch.float64, device="cuda"); w = torch.zeros(64, dtype=torch.float64, device="cuda")
    out = torch.full((34,), 7.0, dtype=torch.float64, device="cuda")
    s = C.c_void_p(int(torch.cuda.current_stream().cuda_stream))
    vp = lambda t: C.c_void_p(int(t.data_ptr()))
    for k, n, ldv in ((33, 64, 64), (0, 64, 64), (4, 0, 64), (4, (1 << 40) + 1, (1 << 40) + 1), (4, 64, 63)):
        rc = L.dmrg_gemv_trans_static(vp(V), ldv, n, k, vp(w), vp(out), s)
        assert rc == lib.DMRG_E_INVALID_ARG, (k, n, ldv, rc)
        assert b"gemv_trans_static" in L.dmrg_last_error(None)
    assert b"ldv" in L.dmrg_last_error(None)
    rc = L.dmrg_gemv_trans_static(vp(V), 64, 64, 33, vp(w), vp(out), s)
    assert rc == lib.DMRG_E_INVALID_ARG and b"33" in L.dmrg_last_error(None) and b"32" in L.dmrg_last_error(None)
    assert L.dmrg_gemv_trans_static(None, 64, 64, 4, vp(w), vp(out), s) == lib.DMRG_E_INVALID_ARG
    torch.cuda.synchronize()
    assert torch.all(out == 7.0)                               # nothing was launched
    with pytest.raises(lib.DmrgError):
        lib.gemv_trans_static(V, 33, w, out)
