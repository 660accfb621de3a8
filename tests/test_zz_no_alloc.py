"""hb_moments_static (-m gpu): the standalone moments pass with its scratch in a static device array of libhb.so, for
callers that cannot allocate device memory (include/hb.h).  Collected last on purpose (file name): the suite runs
with `pytest -x`, and a failure here must not hide any other test.

Checked against the existing path hb_moments (caller-owned scratch) with the bounds of
tests/test_gpu_parity.py::test_standalone_moments (means rtol 1e-12, second moments 1e-9 of sigma_i sigma_j) -- and,
since both paths launch the same kernels on the same grid in the same order, bit for bit -- on two calls in a row; the
second bunch is smaller than the first, so rows of the shared array that still hold the first call's partials must not
be read.  The oracle is the third witness.
"""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hb():
    import torch
    assert torch.cuda.is_available()
    import paper_2402_17248_b200 as hb
    hb.lib()
    return hb


def sym(rec):
    C = np.zeros((6, 6))
    k = 6
    for i in range(6):
        for j in range(i, 6):
            C[i, j] = C[j, i] = rec[k]
            k += 1
    return C


def close(rec, ref):
    assert np.allclose(rec[:6], ref[:6], rtol=1e-12, atol=1e-18)
    C, R = sym(rec), sym(ref)
    sd = np.sqrt(np.diag(R))
    assert np.max(np.abs(C - R) / np.outer(sd, sd)) < 1e-9


def test_static_scratch_moments_two_calls_in_a_row(hb):
    import torch
    torch.cuda.set_device(0)
    out = torch.empty(27, dtype=torch.float64, device="cuda:0")             # the caller's output buffer
    bunches = []
    for n, seed, shift in ((1_000_003, 31, 1e-3), (40_001, 32, -2e-3)):      # many blocks, then few; both ragged
        x = wl.gaussian_bunch(n, seed) + (np.arange(6, dtype=np.float32)[:, None] * np.float32(shift))
        bunches.append((x, hb.to_device(x), list(np.arange(6) * shift)))
    existing = [hb.moments(c, pivot=pv).cpu().numpy() for _, c, pv in bunches]   # hb_moments, caller-owned scratch
    torch.cuda.synchronize()
    for k, (x, c, pv) in enumerate(bunches):
        out.fill_(float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(0)[0]
        hb.moments_static(c, out, pivot=pv)                                  # nothing of torch's runs in between
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info(0)[0]
        rec = out.cpu().numpy()
        close(rec, existing[k])
        assert np.array_equal(rec, existing[k])                              # same kernels, same grid, same order
        close(rec, oracle.moments(np.ascontiguousarray(x.astype(np.float64))))
        assert np.array_equal(hb.to_host(c), x)                              # read-only
        # the second call finds everything in place (the first one may have made the driver load the module): the
        # device's free memory does not shrink across it -- no cudaMalloc behind the entry point
        if k == 1:
            assert free_after >= free_before


def test_static_scratch_moments_without_pivot_and_empty(hb):
    import torch
    out = torch.empty(27, dtype=torch.float64, device="cuda:0")
    x = wl.gaussian_bunch(4096, 33)
    c = hb.to_device(x)
    hb.moments_static(c, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), hb.moments(c).cpu().numpy())
    hb.hb_moments_static(*[c[j].data_ptr() for j in range(6)], 0, None, out.data_ptr(),
                         torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.all(np.isnan(out.cpu().numpy()))                               # n = 0: a record of NaNs, as hb_moments


def test_static_scratch_moments_rejects_sizes_beyond_its_maximum(hb):
    import torch
    limit = hb.hb_moments_static_max_particles()
    assert limit == 2 ** 28
    out = torch.zeros(27, dtype=torch.float64, device="cuda:0")
    c = hb.to_device(wl.gaussian_bunch(1024, 34))
    ptrs = [c[j].data_ptr() for j in range(6)]
    with pytest.raises(hb.HbError) as err:                                   # refused before anything is touched
        hb.hb_moments_static(*ptrs, limit + 1, None, out.data_ptr(), 0)
    assert "HB_ERR_INVALID_ARG" in str(err.value) and "HB_MOMENTS_STATIC_MAX_N" in str(err.value)
    with pytest.raises(hb.HbError):
        hb.hb_moments_static(*ptrs, 1024, None, 0, 0)                        # NULL output
    with pytest.raises(hb.HbError):
        hb.hb_moments_static(ptrs[0] + 4, *ptrs[1:], 1024, None, out.data_ptr(), 0)   # misaligned array
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy() == 0.0)
