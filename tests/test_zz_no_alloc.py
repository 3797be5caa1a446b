"""vr_volume_histogram_noalloc: the histogram entry point for callers that cannot allocate device memory.

Two kinds of user of this library are in that position.  One runs the renderer inside a process whose own allocator
(PyTorch's caching allocator, an RMM pool) has taken nearly all of the GPU, so a cudaMalloc made by the library behind
that allocator's back fails although the application has room.  The other has frames in flight on other streams and
cannot afford vr_volume_histogram's cudaFree, which waits for the whole device.  For them the bins live in a fixed
array inside libvr_b200.so (4096 bins + the NaN counter = 32 776 bytes per GPU, held until the process ends).

What is checked: the counts equal vr_volume_histogram's bit for bit (integers: the tolerance every histogram test
here uses is zero), on calls made back to back — the array keeps what the previous call left in it, so a second call
with fewer bins, another range or another cube would show stale counts if the entry point did not clear what it uses.
The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process and after the other GPU tests.
"""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def vr():
    from paper_1008_0135_b200 import build as vr_build
    vr_build.build()
    from paper_1008_0135_b200 import vr as binding
    binding.lib()                      # fails loudly if libvr_b200.so is missing: no fallback
    return binding


def test_noalloc_rejects_bad_arguments_without_device(vr):
    """Argument checks come before anything touches a GPU."""
    L = vr.lib()
    counts = (C.c_longlong * 8)()
    assert L.vr_volume_histogram_noalloc(None, 8, 0.0, 1.0, counts, None) == vr.VR_ERR_INVALID_ARG
    assert "NULL" in vr.vr_last_error()


@pytest.mark.gpu
def test_noalloc_histogram_equals_allocating_path_on_consecutive_calls(vr):
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    g = torch.Generator(device="cuda").manual_seed(11)
    cube_a = torch.randn((33, 70, 130), generator=g, device="cuda") * 3.0 + 1.0
    cube_a[0, 0, 0] = float("nan"); cube_a[32, 69, 129] = float("nan")
    cube_b = torch.rand((19, 35, 61), generator=g, device="cuda") * 10.0 - 5.0
    vol_a, vol_b = vr.Volume(cube_a), vr.Volume(cube_b)
    try:
        # back to back, each call leaving its counts in the shared array for the next one to trip over:
        # most bins first, then fewer bins over another range, then another cube, then the first case again
        calls = [(vol_a, 4096, -4.0, 7.5), (vol_a, 64, -1.0, 2.0), (vol_b, 1000, -5.0, 5.0), (vol_b, 1, 0.0, 1.0),
                 (vol_a, 4096, -4.0, 7.5), (vol_a, 4096, -4.0, 7.5)]
        got = [v.vr_volume_histogram_noalloc(n, lo, hi) for v, n, lo, hi in calls]
        for (v, n, lo, hi), (counts, n_nan) in zip(calls, got):
            want, want_nan = v.vr_volume_histogram(n, lo, hi)
            assert n_nan == want_nan == (2 if v is vol_a else 0)
            assert counts.dtype == want.dtype and counts.shape == want.shape
            assert np.array_equal(counts, want), (n, lo, hi)
            assert counts.sum() + n_nan == int(np.prod(v.dims))
        # and against numpy's count of the same float32 bin expression, so that "equal" is not "equally wrong"
        counts, _ = vol_b.vr_volume_histogram_noalloc(100, -5.0, 5.0)
        x = cube_b.cpu().numpy().reshape(-1)
        b = np.floor((x - np.float32(-5.0)) * (np.float32(100) / (np.float32(5.0) - np.float32(-5.0))))
        assert np.array_equal(counts, np.bincount(np.clip(b, 0, 99).astype(np.int64), minlength=100))

        # the array cannot grow: more bins than it holds is an error that says so, and nothing is written
        with pytest.raises(vr.VrError) as e:
            vol_a.vr_volume_histogram_noalloc(4097, -4.0, 7.5)
        assert e.value.status == vr.VR_ERR_INVALID_ARG and "4096" in str(e.value)
        for bad in [(0, 0.0, 1.0), (16, 1.0, 1.0), (16, 0.0, float("inf"))]:
            with pytest.raises(vr.VrError) as e:
                vol_a.vr_volume_histogram_noalloc(*bad)
            assert e.value.status == vr.VR_ERR_INVALID_ARG
        # a refused call leaves the next good one untouched
        counts, n_nan = vol_a.vr_volume_histogram_noalloc(64, -1.0, 2.0)
        want, want_nan = vol_a.vr_volume_histogram(64, -1.0, 2.0)
        assert n_nan == want_nan and np.array_equal(counts, want)
    finally:
        vol_a.close()
        vol_b.close()
