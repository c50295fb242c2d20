"""`-m gpu` test of u1mps_expect_n_all_static (include/u1mps.h): step a6 on the library's static device scratch, for
callers that must not allocate.  Collected last on purpose (the suite runs with `pytest -x`).  The reference is the
existing path, u1mps_expect_n_all, on the same handle; tolerance 1e-9 as for every <n_k> comparison of the parity tests
(the two run the same kernel with the same slice count, so they are in fact bit-identical)."""
import ctypes as C
import dataclasses

import numpy as np
import pytest

from gpu_helpers import make_gpu
from paper_2303_11409_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-9


def _advance(gpu, w, columns):
    for sites, us in columns:
        gpu.apply_gate_column(sites, us, cutoff=w.cutoff)


def test_static_scratch_matches_the_arena_path_on_two_calls_in_a_row():
    import torch
    w = dataclasses.replace(inputs.WORKLOADS[2], chi=24)        # M = 64, truncating: sectors of many sizes
    cols = list(inputs.gate_columns(w, 8))
    gpu = make_gpu(w.M, w.d, w.N, w.chi)
    gpu.set_product_state(w.occ)
    _advance(gpu, w, cols[:5])
    out1 = torch.full((w.M,), float("nan"), dtype=torch.float64, device="cuda")
    out2 = torch.full((w.M,), float("nan"), dtype=torch.float64, device="cuda")
    out3 = torch.full((w.M,), float("nan"), dtype=torch.float64, device="cuda")
    launches0 = gpu.launch_count()

    # call 1 and call 2 back to back on the same state: the second one finds the array as the first one left it
    gpu.expect_n_all_static(out1)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    gpu.expect_n_all_static(out2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before          # nothing was allocated on the device
    assert gpu.launch_count() == launches0 + 2                   # one kernel per call
    ref = gpu.expect_n_all()
    for out in (out1, out2):
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert np.max(np.abs(got - ref)) <= TOL
    assert np.array_equal(out1.cpu().numpy(), out2.cpu().numpy())   # the sums are added in a fixed order

    # call 3 after the state has moved on: a fresh result, not the previous one
    _advance(gpu, w, cols[5:])
    gpu.expect_n_all_static(out3)
    torch.cuda.synchronize()
    ref3 = gpu.expect_n_all()
    assert np.max(np.abs(out3.cpu().numpy() - ref3)) <= TOL
    assert np.max(np.abs(ref3 - ref)) > 1e-6                     # the state did change


def test_static_scratch_is_shared_between_handles_of_different_length():
    import torch
    big = dataclasses.replace(inputs.WORKLOADS[2], chi=16)      # M = 64
    small = inputs.WORKLOADS[1]                                  # M = 16: more slices per site, fewer counters
    res = {}
    for w in (big, small, big):
        gpu = make_gpu(w.M, w.d, w.N, w.chi)
        gpu.set_product_state(w.occ)
        _advance(gpu, w, inputs.gate_columns(w, 4))
        out = torch.full((w.M,), float("nan"), dtype=torch.float64, device="cuda")
        gpu.expect_n_all_static(out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.max(np.abs(got - gpu.expect_n_all())) <= TOL
        res.setdefault(w.name + str(w.chi), []).append(got)
    a, b = res[big.name + "16"]
    assert np.array_equal(a, b)                                  # deterministic whatever the array held before


def test_static_scratch_rejects_what_it_cannot_take():
    import torch
    from paper_2303_11409_b200.binding import ETOOBIG, STATIC_SITES_MAX, U1MPSError
    M = STATIC_SITES_MAX + 1
    occ = [1] + [0] * (M - 1)
    gpu = make_gpu(M, 2, 1, 2)
    gpu.set_product_state(occ)
    out = torch.zeros(M, dtype=torch.float64, device="cuda")
    with pytest.raises(U1MPSError) as ei:
        gpu.expect_n_all_static(out)
    assert ei.value.code == ETOOBIG
    assert "maximum" in str(ei.value)
    assert abs(np.sum(gpu.expect_n_all()) - 1.0) <= TOL         # the handle is still usable; the arena path takes M = 1025

    ok = make_gpu(STATIC_SITES_MAX, 2, 1, 2)                     # exactly the maximum is accepted
    ok.set_product_state([1] + [0] * (STATIC_SITES_MAX - 1))
    out = torch.full((STATIC_SITES_MAX,), float("nan"), dtype=torch.float64, device="cuda")
    ok.expect_n_all_static(out)
    torch.cuda.synchronize()
    assert np.max(np.abs(out.cpu().numpy() - ok.expect_n_all())) <= TOL

    host = np.zeros(STATIC_SITES_MAX)                            # a host pointer is refused, not dereferenced
    r = ok.lib.u1mps_expect_n_all_static(ok.h, C.c_void_p(host.ctypes.data))
    assert r == -1
    assert ok.lib.u1mps_expect_n_all_static(ok.h, None) == -1
