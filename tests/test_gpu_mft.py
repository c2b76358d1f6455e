"""Fraunhofer matrix Fourier transform on the GPU (fresnel_mft), run
with -m gpu: two complex GEMMs on the FP64 tensor cores against the oracle's plain definition (oracle.mft, pinned by
P24-P26), whole field, north-star tolerances + max-abs bound; sizes that are not multiples of the GEMM tiles."""
import numpy as np
import pytest

from test_gpu_parity import TOL, assert_parity, field, to_dev

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
@pytest.mark.parametrize("na,nb", [(64, 64), (128, 37), (100, 130), (512, 200), (1024, 256)])
@pytest.mark.parametrize("direction", [+1, -1])
def test_mft_matches_the_oracle(torch_cuda, B, oracle, na, nb, dtype, direction):
    """Output grids finer and coarser than critical, nb below and above na, two wavelengths per call."""
    torch = torch_cuda
    u = field(na, 13000 + na + nb, 2, dtype)
    dx = np.array([1.5e-5, 1.2e-5])
    lam = np.array([0.8e-6, 0.65e-6])
    f = 0.6
    dxo = lam * f / (na * dx) * np.array([0.31, 1.7])
    plan = B.Plan(na, 2, dtype)
    d = to_dev(torch, u, dtype)
    out = torch.zeros(2, nb, nb, dtype=d.dtype, device="cuda")
    plan.mft(d, out, dx, dxo, lam, f, direction)
    want = np.stack([oracle.mft(u[b], dx[b], nb, dxo[b], lam[b], f, direction) for b in range(2)])
    assert_parity(out.cpu().numpy(), want, dtype)
    assert np.array_equal(d.cpu().numpy().reshape(u.shape).astype(np.complex128), u)      # the input is read only


def test_mft_is_the_fourier_core_of_direct_fresnel_and_round_trips(torch_cuda, B, oracle):
    """On the GPU too: at critical sampling chirp x MFT x chirp equals fresnel_propagate_direct, and the inverse
    direction undoes the forward one."""
    torch = torch_cuda
    na, dx, lam, z = 256, np.array([2e-5]), np.array([1e-6]), 0.35
    u = field(na, 13100, 1)
    plan = B.Plan(na, 1, "c128")
    a = to_dev(torch, u, "c128")
    px = plan.propagate_direct(a, dx, lam, z)
    b = to_dev(torch, u, "c128")
    plan.apply_qpf(b, dx, lam, z)
    out = torch.zeros_like(b)
    plan.mft(b, out, dx, px, lam, z, +1)
    plan.apply_qpf(out, px, lam, z)
    assert np.linalg.norm(out.cpu().numpy() - a.cpu().numpy()) / np.linalg.norm(a.cpu().numpy()) <= 1e-11
    c = to_dev(torch, u, "c128")
    fwd = torch.zeros_like(c)
    back = torch.zeros_like(c)
    plan.mft(c, fwd, dx, px, lam, z, +1)
    plan.mft(fwd, back, px, dx, lam, z, -1)
    assert np.linalg.norm(back.cpu().numpy().reshape(na, na) - u[0]) / np.linalg.norm(u[0]) <= 1e-11


def test_mft_errors_and_graph_capture(torch_cuda, B, oracle):
    torch = torch_cuda
    na, nb = 128, 48
    u = field(na, 13200, 1)
    s = torch.cuda.Stream()
    plan = B.Plan(na, 1, "c128", stream=s)
    d = to_dev(torch, u, "c128")
    out = torch.zeros(1, nb, nb, dtype=d.dtype, device="cuda")
    with pytest.raises(B.FresnelError):
        plan.mft(d, out, [1e-5], [1e-5], [1e-6], 0.0)
    with pytest.raises(B.FresnelError):
        plan.mft(d, out, [1e-5], [-1e-5], [1e-6], 0.5)
    plan.reserve_mft(nb)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            plan.mft(d, out, [1e-5], [2e-5], [1e-6], 0.5)
    g.replay()
    torch.cuda.synchronize()
    want = oracle.mft(u[0], 1e-5, nb, 2e-5, 1e-6, 0.5, +1)
    assert_parity(out.cpu().numpy(), want[None], "c128")
