"""GPU test of jerk_prepare_spectrum_static, the spectrum-preparation entry point that allocates no device memory.

Who needs it: code that calls this library from a place where cudaMalloc is not an option -- a host framework whose
own pool owns the GPU's memory and forbids side allocations, an acquisition loop that cannot afford the allocator's
lock and implicit synchronisation, a plug-in that is handed an input and an output buffer and nothing else.  Such a
caller cannot produce the d_scratch that jerk_prepare_spectrum wants, so the library keeps that intermediate array in
its own image (8 MiB per GPU, at most 2^21 samples per call; include/jerk.h).

What is checked: the new entry point gives the same spectrum as the existing caller-scratch path, within the
tolerance of tests/test_gpu_spectrum.py, on two calls in a row -- the second one shorter than the first and on
different data, so that it runs on top of whatever the first call left in the shared array -- and then once more at
the first size; sizes above the limit are refused with JERK_ELIMIT and a message that names the limit.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  Nothing here depends on the other tests having run (or not): it passes alone in a fresh process, where
its first call is the one that does the per-device address look-up, and after the whole suite."""
import numpy as np
import pytest

from paper_1911_01353_b200 import binding, build

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

TOL = 2e-5      # tests/test_gpu_spectrum.py: |X - X_ref| <= TOL * max(1, |X_ref|)


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    binding.load_library()


def _series(log2n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    x = rng.standard_normal(1 << log2n, dtype=np.float32)
    x += 0.5 * np.cos(2 * np.pi * 0.0137 * np.arange(x.size)).astype(np.float32)
    return torch.from_numpy(x).cuda()


def _close(got, ref):
    g = got.cpu().numpy().view(np.complex64).reshape(-1).astype(np.complex128)
    r = ref.cpu().numpy().view(np.complex64).reshape(-1).astype(np.complex128)
    assert np.isfinite(g.view(np.float64)).all()
    err = np.abs(g - r) / np.maximum(1.0, np.abs(r))
    assert err.max() <= TOL, (err.max(), int(err.argmax()))


def test_two_calls_in_a_row_match_the_caller_scratch_path():
    """Largest allowed size, then a short series straight after it on the same stream (no synchronisation in between),
    then the large size again: each result equals jerk_prepare_spectrum's."""
    big = _series(21, 19110135)                  # 2^21 samples = the limit: the whole static array is in use
    small = _series(14, 19110136)                # 2^14: runs over the first 64 KiB of what the big call left behind
    out_big = torch.full((big.numel() // 2, 2), float("nan"), dtype=torch.float32, device="cuda")
    out_small = torch.full((small.numel() // 2, 2), float("nan"), dtype=torch.float32, device="cuda")
    binding.prepare_spectrum_static(big, 1000, d_spec=out_big)
    binding.prepare_spectrum_static(small, 1000, d_spec=out_small)
    torch.cuda.synchronize()
    ref_big = binding.prepare_spectrum(big, 1000, mode="mean")
    ref_small = binding.prepare_spectrum(small, 1000, mode="mean")
    torch.cuda.synchronize()
    _close(out_big, ref_big)
    _close(out_small, ref_small)
    out_again = torch.full_like(out_big, float("nan"))
    binding.prepare_spectrum_static(big, 1000, d_spec=out_again)
    torch.cuda.synchronize()
    _close(out_again, ref_big)


def test_the_call_allocates_no_device_memory():
    """Free device memory as the driver reports it is the same before and after a call whose buffers already exist."""
    x = _series(20, 19110137)
    out = torch.empty((x.numel() // 2, 2), dtype=torch.float32, device="cuda")
    binding.prepare_spectrum_static(x, 1000, d_spec=out)      # first use on this device (if run alone): set-up happens here
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        binding.prepare_spectrum_static(x, 1000, d_spec=out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before


def test_sizes_above_the_limit_are_refused():
    lib = binding.load_library()
    assert binding.STATIC_SPECTRUM_MAX_SAMPLES == 1 << 21
    n = 1 << 22
    x = torch.zeros(n, dtype=torch.float32, device="cuda")
    out = torch.full((n // 2, 2), 7.0, dtype=torch.float32, device="cuda")
    import ctypes as C
    rc = lib.jerk_prepare_spectrum_static(C.c_void_p(x.data_ptr()), n, 1000, C.c_void_p(out.data_ptr()), None)
    assert rc == binding.JERK_ELIMIT
    msg = lib.jerk_strerror(rc).decode()
    assert "2^21" in msg and "jerk_prepare_spectrum" in msg
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                 # refused before any launch: the output is untouched
    with pytest.raises(binding.JerkError) as ei:
        binding.prepare_spectrum_static(x, 1000, d_spec=out)
    assert ei.value.status == binding.JERK_ELIMIT
