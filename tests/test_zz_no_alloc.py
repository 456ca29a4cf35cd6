"""bg_amplitudes_host_noalloc: the host-buffer entry point for callers that cannot allocate device memory.

Some users of the library have no device memory to hand over and no way to get any: a plug-in that runs beside
a framework whose memory pool already owns nearly all of HBM (its own cudaMalloc fails), code on a path where
cudaMalloc / cudaFree's device-wide synchronisation is not acceptable, or a plain C / Fortran program that only
has host arrays.  For them the library carries its staging area inside its own image (a fixed 8 MiB __device__
array) and this entry point allocates nothing at call time.  The price is a limit on the batch per call
(bg_noalloc_max_batch) and one shared array: calls that overlap on the GPU race, calls in a row do not.

This file is named so that pytest collects it LAST: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  The test is self-contained (own inputs, no state from other tests) and passes
both alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2502_07060_b200 import build, inputs


@pytest.fixture(scope="module")
def bgl():
    build.build()
    from paper_2502_07060_b200 import binding
    binding.load()
    return binding


def test_limit_is_stated_by_the_library(bgl):
    """host-only calls: the fixed array's size and what fits into it (momenta | polarisations | out | status,
    each rounded up to 256 bytes)"""
    assert bgl.bg_noalloc_scratch_bytes() == 8 << 20
    for field, n, d, w in [(0, 8, 6, 4), (1, 6, 4, 16), (0, 16, 16, 4), (1, 16, 16, 16), (1, 12, 6, 16)]:
        def need(b):
            r = lambda x: (x + 255) // 256 * 256
            return 2 * r(b * n * d * w) + r(b * w) + r(b * 4)
        m = bgl.bg_noalloc_max_batch(field, n, d)
        assert m > 1000 and need(m) <= 8 << 20 < need(m + 1)
    assert bgl.bg_noalloc_max_batch(0, 8, 6) == 21398
    assert bgl.bg_noalloc_max_batch(2, 8, 6) == 0          # a generic prime needs bg_evaluate
    assert bgl.bg_noalloc_max_batch(0, 3, 6) == 0
    assert "bg_noalloc_max_batch" in bgl.bg_status_string(bgl.BG_ERR_TOO_LARGE)


def _existing_path(bgl, mom, pol):
    """the path the library already had: device tensors from torch, bg_amplitudes_status on torch's stream"""
    import torch
    dm, dp = bgl.to_device(mom), bgl.to_device(pol)
    status = torch.full((mom.shape[0],), -1, dtype=torch.int32, device="cuda")
    out = bgl.amplitudes(dm, dp, status=status)
    torch.cuda.synchronize()
    return bgl.to_numpy(out), bgl.to_numpy(status)


@pytest.mark.gpu
@pytest.mark.parametrize("field,n,d", [("fp31", 8, 6), ("c128", 6, 4)])
def test_two_calls_in_a_row_match_the_existing_path(bgl, field, n, d):
    """Two calls back to back through the shared array, the second smaller and on other inputs (so the array
    still holds the first call's bytes behind it), each compared with the existing device-buffer path on the
    same inputs: bit-exact over F_p, and within the first branch of rule R9 (1e-10 relative) over complex128
    -- the same kernel runs in both, so the difference is in fact zero."""
    f = bgl.FIELD_FP31 if field == "fp31" else bgl.FIELD_C128
    top = bgl.bg_noalloc_max_batch(f, n, d)
    for batch, seed in [(top, 101), (top // 3 + 7, 202)]:
        mom, pol, _ = inputs.make_inputs(field, n, d, batch, seed=seed)
        status = np.full(batch, 0xFFFFFFFF, dtype=np.uint32)
        out = np.empty(batch, dtype=mom.dtype)
        got = bgl.amplitudes_host_noalloc(mom, pol, out=out, status=status)
        assert got is out
        ref, ref_status = _existing_path(bgl, mom, pol)
        if field == "fp31":
            assert np.array_equal(out, ref)
        else:
            assert np.all(np.abs(out - ref) <= 1e-10 * np.abs(ref))
        assert np.array_equal(status, ref_status)


@pytest.mark.gpu
def test_too_large_is_refused_before_anything_runs(bgl):
    f, n, d = bgl.FIELD_FP31, 8, 6
    batch = bgl.bg_noalloc_max_batch(f, n, d) + 1
    mom, pol, _ = inputs.make_inputs("fp31", n, d, batch, seed=5)
    out = np.full(batch, 0xDEADBEEF, dtype=np.uint32)
    rc = bgl.bg_amplitudes_host_noalloc(f, n, d, batch, mom.ctypes.data, pol.ctypes.data, out.ctypes.data, None, 0)
    assert rc == bgl.BG_ERR_TOO_LARGE
    assert (out == 0xDEADBEEF).all()
    with pytest.raises(bgl.BgError, match="bg_noalloc_max_batch"):
        bgl.amplitudes_host_noalloc(mom, pol)
    # and the call still works afterwards, without a status array
    res = bgl.amplitudes_host_noalloc(mom[:1000], pol[:1000])
    ref, _ = _existing_path(bgl, np.ascontiguousarray(mom[:1000]), np.ascontiguousarray(pol[:1000]))
    assert np.array_equal(res, ref)
    assert bgl.bg_amplitudes_host_noalloc(f, n, d, 0, None, None, None, None, 0) == bgl.BG_OK      # empty batch
    assert bgl.bg_amplitudes_host_noalloc(f, n, d, 8, None, pol.ctypes.data, out.ctypes.data, None, 0) == bgl.BG_ERR_ARG
    assert bgl.bg_amplitudes_host_noalloc(2, n, d, 8, mom.ctypes.data, pol.ctypes.data, out.ctypes.data, None, 0) == bgl.BG_ERR_ARG
