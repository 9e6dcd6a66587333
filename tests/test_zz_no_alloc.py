"""-m gpu test of srpp_mbp_static, the one entry point that allocates no device memory (its scratch is a static
__device__ array inside libsrpp.so; include/srpp.h).  Collected last on purpose (the file name sorts after every other
test file): the suite runs with pytest -x, so a failure here must not hide the other tests.

The new entry point is compared with the existing path (srpp_mbp through binding.Solver.mbp, caller-owned workspace) on
the same inputs, within the tolerance the MBP parity tests use, on two calls in a row -- the second on a smaller,
different input, so that contents the first call left in the shared array would show -- and then on the first input
again.  Passes alone in a fresh process and after the other tests (the array is per process and every call clears what
it needs)."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _halos(seed, sizes, eps_spread=1.0):
    rng = np.random.default_rng(seed)
    tot = int(sum(sizes))
    hs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    pos = np.empty((tot, 4), dtype=np.float32)
    centres = np.repeat(rng.uniform(5.0, 60.0, (len(sizes), 3)), sizes, axis=0)
    pos[:, :3] = (centres + rng.normal(0.0, eps_spread, (tot, 3))).astype(np.float32)
    pos[:, 3] = rng.uniform(0.5, 2.0, tot).astype(np.float32)
    return pos, hs


def _compare(torch, binding, pos, hs, eps, label):
    """Existing path vs srpp_mbp_static on one input; returns the free device memory seen around the static call."""
    n, nh = pos.shape[0], len(hs) - 1
    d = torch.from_numpy(pos).cuda()
    sol = binding.Solver((64.0,) * 3, (10,) * 3, 3.0, eps, n_max=16)
    idx0, pmin0, phi0 = sol.mbp(d, hs)                       # existing path: caller-owned workspace
    torch.cuda.synchronize()
    idx1 = torch.full((max(nh, 1),), -7, dtype=torch.int64, device="cuda")[:nh]
    pmin1 = torch.full((max(nh, 1),), float("nan"), dtype=torch.float32, device="cuda")[:nh]
    phi1 = torch.full((max(n, 1),), float("nan"), dtype=torch.float32, device="cuda")[:n]
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    binding.mbp_static(d, hs, eps, idx1, pmin1, phi1)        # new path: the library's static scratch array
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    idx0, pmin0, phi0 = idx0.cpu().numpy(), pmin0.cpu().numpy(), phi0.cpu().numpy()
    idx1, pmin1, phi1 = idx1.cpu().numpy(), pmin1.cpu().numpy(), phi1.cpu().numpy()
    member = np.zeros(n, dtype=bool)
    for h in range(nh):
        member[hs[h]:hs[h + 1]] = True
    # tolerance of the MBP parity tests (tests/test_gpu_parity.py::_mbp_check): 2e-5 of the potential + 1e-6.  Both paths
    # run the same kernels; only the order of the fp64 atomic folds differs.
    assert np.all(np.isfinite(phi1[member])), label
    scale = np.maximum(np.abs(phi0), 1e-30)
    assert np.all(np.abs(phi1[member] - phi0[member]) <= 2e-5 * scale[member] + 1e-6), label
    for h in range(nh):
        if hs[h + 1] == hs[h]:
            assert idx1[h] == -1 and pmin1[h] == 0.0, (label, h)
            continue
        assert hs[h] <= idx1[h] < hs[h + 1], (label, h)
        # the two argmins agree, or differ only between members whose potentials tie within the tolerance
        assert idx1[h] == idx0[h] or abs(phi0[idx1[h]] - phi0[idx0[h]]) <= 4e-5 * abs(phi0[idx0[h]]) + 1e-6, (label, h)
        assert abs(pmin1[h] - pmin0[h]) <= 4e-5 * abs(pmin0[h]) + 1e-6, (label, h)
    print("%s: n=%d halos=%d max |dphi|/|phi| = %.2e, argmin equal in %d of %d halos"
          % (label, n, nh, float(np.max(np.abs(phi1[member] - phi0[member]) / scale[member])) if member.any() else 0.0,
             int(np.sum(idx1 == idx0)), nh))
    return free_before, free_after


def test_mbp_static_matches_existing_path_two_calls_in_a_row():
    import torch
    from paper_1411_3396_b200 import binding
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    binding.load()
    eps = 0.05
    # call 1: several source chunks and target tiles per halo, an empty halo, a ragged tail
    pos_a, hs_a = _halos(11, [70000, 1, 0, 2049, 300, 40, 5003])
    _compare(torch, binding, pos_a, hs_a, eps, "call 1")
    # call 2, right after: smaller and different -- stale accumulators / halo table of call 1 would show
    pos_b, hs_b = _halos(12, [900, 129, 0, 33], eps_spread=0.3)
    fb, fa = _compare(torch, binding, pos_b, hs_b, eps, "call 2")
    assert fa >= fb, "srpp_mbp_static must not allocate device memory (free memory fell by %d bytes)" % (fb - fa)
    # and the first input again
    fb, fa = _compare(torch, binding, pos_a, hs_a, eps, "call 3")
    assert fa >= fb, "srpp_mbp_static must not allocate device memory (free memory fell by %d bytes)" % (fb - fa)


def test_mbp_static_rejects_sizes_beyond_its_array():
    import torch
    from paper_1411_3396_b200 import binding
    lib = binding.load()
    d = torch.zeros((16, 4), dtype=torch.float32, device="cuda")
    idx = torch.empty(4, dtype=torch.int64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    i64 = C.c_int64
    # above the member / halo maxima: LIMIT (-7), decided before any pointer is touched
    n_big = binding.MBP_STATIC_MAX_N + 1
    hs = (i64 * 2)(0, n_big)
    assert lib.srpp_mbp_static(d.data_ptr(), n_big, hs, 1, C.c_float(0.1), None, idx.data_ptr(), None, st) == -7
    nh_big = binding.MBP_STATIC_MAX_HALOS + 1
    hs2 = (i64 * (nh_big + 1))(*([0] * (nh_big + 1)))
    assert lib.srpp_mbp_static(d.data_ptr(), 16, hs2, nh_big, C.c_float(0.1), None, idx.data_ptr(), None, st) == -7
    assert "limit" in binding.strerror(-7)
    # invalid arguments: eps, misaligned positions, halo table beyond n / not monotone
    ok = (i64 * 2)(0, 16)
    assert lib.srpp_mbp_static(d.data_ptr(), 16, ok, 1, C.c_float(0.0), None, idx.data_ptr(), None, st) == -1
    assert lib.srpp_mbp_static(d.data_ptr() + 4, 15, ok, 1, C.c_float(0.1), None, idx.data_ptr(), None, st) == -1
    assert lib.srpp_mbp_static(d.data_ptr(), 16, (i64 * 2)(0, 17), 1, C.c_float(0.1), None, idx.data_ptr(), None, st) == -1
    assert lib.srpp_mbp_static(d.data_ptr(), 16, (i64 * 3)(0, 9, 5), 2, C.c_float(0.1), None, idx.data_ptr(), None, st) == -1
    # exactly at the member maximum is accepted (one halo of 2^20 coincident particles would take long: many small halos)
    n_max = binding.MBP_STATIC_MAX_N
    sizes = [64] * (n_max // 64)
    hs3 = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    big = torch.rand((n_max, 4), generator=g, device="cuda")
    idx3 = torch.empty(len(sizes), dtype=torch.int64, device="cuda")
    binding.mbp_static(big, hs3, 0.1, idx3)
    torch.cuda.synchronize()
    i3 = idx3.cpu().numpy()
    assert np.all((i3 >= hs3[:-1]) & (i3 < hs3[1:]))
