"""fresnel_mft_noalloc (run with -m gpu; collected LAST on purpose): the matrix Fourier transform for callers that may not
allocate device memory -- no plan, scratch in a fixed `static __device__` array inside the library -- against the existing
path (Plan.mft, which the oracle covers in tests/test_gpu_mft.py) on the same inputs, at the tolerances of the other GPU
tests (tests/test_gpu_parity.py: relative L2 <= 1e-11 complex128 / 2e-5 complex64 plus the max-abs bound), on two calls
in a row that share the array (the second with another geometry, so stale contents of the first would show), and the
refusal of problems beyond the array."""
import ctypes

import numpy as np
import pytest

from test_gpu_parity import assert_parity, field, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B(torch_cuda):
    from paper_1806_06467_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_mft_noalloc_equals_the_plan_path_on_two_calls_in_a_row(torch_cuda, B, dtype):
    torch = torch_cuda
    cdt = torch.complex128 if dtype == "c128" else torch.complex64
    lam, f = np.array([0.8e-6, 0.65e-6]), 0.7
    # (na, nb, oversampling of the output grid, direction): 2 * 128 * 512 = 131072 and 2 * 200 * 300 = 120000 <= 262144 elements
    calls = [(512, 128, 3.0, +1), (300, 200, 1.0, -1)]
    mem0 = None
    for i, (na, nb, over, direction) in enumerate(calls):
        u = field(na, 12000 + na, 2, dtype)
        dx = np.array([1.5e-5, 1.2e-5])
        dxo = lam * f / (na * dx) / over
        src = to_dev(torch, u, dtype)
        plan = B.Plan(na, 2, dtype)
        want = torch.zeros(2, nb, nb, dtype=cdt, device="cuda")
        plan.mft(src, want, dx, dxo, lam, f, direction)
        got = torch.full((2, nb, nb), float("nan"), dtype=cdt, device="cuda")
        torch.cuda.synchronize()
        if i == 1:
            mem0 = torch.cuda.memory_allocated()
        B.mft_noalloc(src, got, dx, dxo, lam, f, direction)
        torch.cuda.synchronize()
        if i == 1:
            assert torch.cuda.memory_allocated() == mem0            # (torch's own allocator saw nothing either)
        assert_parity(got.cpu().numpy().astype(np.complex128), want.cpu().numpy().astype(np.complex128), dtype, f"call {i}")
        assert torch.equal(got, want), "same kernels, same inputs: bit-identical"
        plan.close()


def test_mft_noalloc_refuses_what_does_not_fit(torch_cuda, B):
    torch = torch_cuda
    L = B.lib()
    assert L.fresnel_status_string(5) == b"FRESNEL_ERR_TOO_LARGE"
    src = torch.zeros(1, 1024, 1024, dtype=torch.complex128, device="cuda")
    out = torch.zeros(1, 257, 257, dtype=torch.complex128, device="cuda")
    with pytest.raises(B.FresnelError) as ei:                          # 1024 * 257 > 262144
        B.mft_noalloc(src, out, 1e-5, 1e-5, 1e-6, 1.0)
    assert ei.value.status == 5
    assert B.MFT_NOALLOC_MAX_ELEMS == 262144 and B.MFT_NOALLOC_MAX_BATCH == 32
    small = torch.zeros(33, 16, 16, dtype=torch.complex64, device="cuda")  # batch beyond the scalar block
    with pytest.raises(B.FresnelError) as ei:
        B.mft_noalloc(small, torch.zeros(33, 8, 8, dtype=torch.complex64, device="cuda"), 1e-5, 1e-5, 1e-6, 1.0)
    assert ei.value.status == 5
    # the largest problem that fits runs: one 1024 -> 256 transform
    u = field(1024, 12100, 1, "c128")
    d = to_dev(torch, u, "c128")
    got = torch.zeros(1, 256, 256, dtype=torch.complex128, device="cuda")
    want = torch.zeros_like(got)
    B.mft_noalloc(d, got, 1e-5, 2e-5, 1e-6, 1.0)
    plan = B.Plan(1024, 1, "c128")
    plan.mft(d, want, 1e-5, 2e-5, 1e-6, 1.0)
    torch.cuda.synchronize()
    assert_parity(got.cpu().numpy(), want.cpu().numpy(), "c128", "1024 -> 256")
    # argument errors are INVALID_ARG, not TOO_LARGE
    h = ctypes.c_void_p(d.data_ptr())
    one = (ctypes.c_double * 1)(1e-5)
    assert L.fresnel_mft_noalloc(h, h, 64, 64, 1, 1, one, one, one, 1.0, 1, None) == 1      # in == out
    assert L.fresnel_mft_noalloc(h, ctypes.c_void_p(got.data_ptr()), 64, 64, 1, 1, one, one, one, 0.0, 1, None) == 1
