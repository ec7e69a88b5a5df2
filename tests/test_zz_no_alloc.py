"""-m gpu: cbmf_ifft_noalloc_dev, the inverse FFT for callers that cannot allocate device memory.

Who needs it: code that lives inside another program's memory budget (a plug-in of a framework whose caching
allocator already owns the GPU), an online analysis loop that may not stall in the device-wide synchronisation of
cudaMalloc / cudaFree, and code that runs while a stream of the process is being captured.  Such callers hand in
their input and output arrays; the library's inter-pass buffer, which a context would cudaMalloc, is a fixed 8 MiB
array inside the library image instead -- hence the limit n <= 2^20, and hence ONE buffer per GPU that every call
shares and that still holds whatever the previous call wrote.

What is checked: the entry point against the existing context path (cbmf_debug_ifft_dev, whose parity with the
oracle's FFT is test_gpu_parity.test_ifft_matches_oracle_fft) within that test's tolerance, on calls issued back to
back on one stream WITHOUT a wait in between, with different sizes and data, so that a result depending on the
buffer's stale contents or on a missing order between launch pairs would show; the limit and argument errors; and
that a repeated call leaves the free device memory where it was.

This file is collected last on purpose (pytest -x stops at the first failure: a failure here hides nothing) and
does not depend on the tests before it: it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

REL_TOL = 3e-5          # of the rms of the reference, as test_ifft_matches_oracle_fft (fp32: ~ eps * log2 N * few)


@pytest.fixture(scope="module")
def cbmf():
    from paper_1006_4644_b200 import cbmf as m
    m.lib()
    return m


def _input(torch, seed, batch, n):
    rng = np.random.default_rng(seed)
    x = (rng.standard_normal((batch, n)) + 1j * rng.standard_normal((batch, n))).astype(np.complex64)
    return torch.from_numpy(x).cuda()


def _existing_path(cbmf, x, n):
    """The context path: cbmf_debug_ifft_dev with its cudaMalloc'ed inter-pass buffer."""
    with cbmf.Context(n, 4096.0, 40.0) as g:
        return g.debug_ifft(x).clone()


def _rel_err(got, ref):
    ref = ref.cpu().numpy().astype(np.complex128)
    got = got.cpu().numpy().astype(np.complex128)
    return float(np.max(np.abs(got - ref)) / np.sqrt(np.mean(np.abs(ref) ** 2)))


def test_two_calls_in_a_row_match_the_context_path(cbmf):
    """Three calls queued behind one another, no wait between them: 5 vectors of 2^18 (4 fit the array: two launch
    pairs, the second ragged), then 3 of 2^14 (the array is now full of the first call's data), then 2^18 again
    with new data.  Each must equal what a context computes for the same input."""
    import torch
    cases = [(11, 5, 1 << 18), (12, 3, 1 << 14), (13, 6, 1 << 18)]
    xs = [_input(torch, s, b, n) for s, b, n in cases]
    outs = [torch.full_like(x, float("nan")) for x in xs]
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream().cuda_stream
    for x, out, (_, _, n) in zip(xs, outs, cases):
        assert cbmf.ifft_noalloc_dev(x, out, n, stream) == cbmf.OK
    torch.cuda.synchronize()
    for x, out, (_, b, n) in zip(xs, outs, cases):
        ref = _existing_path(cbmf, x, n)
        for i in range(b):
            err = _rel_err(out[i], ref[i])
            assert err < REL_TOL, (n, i, err)


def test_maximum_size_and_repeat_without_allocation(cbmf):
    """n = CBMF_NOALLOC_MAX_N: one vector fills the whole array, so every vector is its own launch pair.  The call
    is made twice; the second one must not lower the free device memory (a scratch allocation would take 8 MiB)."""
    import torch
    n = cbmf.NOALLOC_MAX_N
    x = _input(torch, 21, 2, n)
    out1, out2 = torch.empty_like(x), torch.empty_like(x)
    stream = torch.cuda.current_stream().cuda_stream
    assert cbmf.ifft_noalloc_dev(x, out1, n, stream) == cbmf.OK       # first call at this size: one-off set-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    assert cbmf.ifft_noalloc_dev(x, out2, n, stream) == cbmf.OK
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert free_before - free_after < (1 << 20), (free_before, free_after)
    ref = _existing_path(cbmf, x, n)
    for out in (out1, out2):
        for i in range(2):
            err = _rel_err(out[i], ref[i])
            assert err < REL_TOL, (i, err)


def test_limit_and_argument_errors(cbmf):
    """Beyond the fixed array the call refuses with its own code and touches nothing; bad arguments are EINVAL."""
    import torch
    n_big = 2 * cbmf.NOALLOC_MAX_N
    x = torch.zeros((1, n_big), dtype=torch.complex64, device="cuda")
    out = torch.full_like(x, 7.0)
    assert cbmf.ifft_noalloc_dev(x, out, n_big) == cbmf.ELIMIT
    assert "scratch" in cbmf.lib().cbmf_strerror(cbmf.ELIMIT).decode()
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
    L = cbmf.lib()
    p, q = x.data_ptr(), out.data_ptr()
    assert L.cbmf_ifft_noalloc_dev(0, None, p, q, 3 << 12, 1) == cbmf.EINVAL        # not a power of two
    assert L.cbmf_ifft_noalloc_dev(0, None, p, q, 1 << 11, 1) == cbmf.EINVAL        # below the two-pass floor
    assert L.cbmf_ifft_noalloc_dev(0, None, p, q, 1 << 12, -1) == cbmf.EINVAL
    assert L.cbmf_ifft_noalloc_dev(0, None, None, q, 1 << 12, 1) == cbmf.EINVAL
    assert L.cbmf_ifft_noalloc_dev(0, None, p + 8, q, 1 << 12, 1) == cbmf.EINVAL    # 16-byte alignment
    assert L.cbmf_ifft_noalloc_dev(torch.cuda.device_count(), None, p, q, 1 << 12, 1) == cbmf.EINVAL
    assert L.cbmf_ifft_noalloc_dev(0, None, None, None, 1 << 12, 0) == cbmf.OK      # nothing to do
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
