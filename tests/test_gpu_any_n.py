"""Grids that are not a power of two ("N = 2800 ran faster than
4096"; :259 npix = 1025), run with -m gpu.  The CUDA path (gen_kernel.cuh: mixed-radix Stockham stages in shared
memory, Bluestein for sizes with a large prime factor; mr_kernel.cuh: the register-resident mixed-radix pass of
N = 700, 1400, 2800) against the oracle's plain O(N^3) separable DFT, whole field, north-star tolerances + the max-abs
bound.  Sizes: 100 = 2^2 5^2, 130 = 2 5 13, 175 = 5^2 7 (odd), 243 = 3^5 (odd), 335 = 5 67 (odd, Bluestein over
M = 672), 360 = 2^3 3^2 5, 488 = 2^3 61 and 1025 = 5^2 41 (odd; one prime 17..61 as a direct first stage), 700 = 2^2 5^2 7
(register-resident: partial butterfly rounds, a partial last TMA box), 1100 = 2^2 5^2 11, 1200 = 3 5 5 16 (register-resident with a
radix-3 stage), 1400 = 2^3 5^2 7, 1500 and 2400 (register-resident in five stages), 2800 = 2^4 5^2 7, 4100 = 2^2 5^2 41 (the paper's
App. B call: npix = 1025 at beam ratio 0.25); every register-resident size also against the shared-memory pass.
"""
import math

import numpy as np
import pytest

from test_gpu_parity import TOL, assert_parity, field, map_dev, map_host, to_dev

pytestmark = pytest.mark.gpu

SIZES = [100, 130, 175, 243, 335, 360, 488, 700, 1025, 1200]


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
@pytest.mark.parametrize("N", SIZES)
@pytest.mark.parametrize("direction,centered", [(+1, False), (-1, False), (+1, True), (-1, True)])
def test_fft2d_any_n(torch_cuda, B, oracle, N, dtype, direction, centered):
    """fresnel_fft2d: forward / inverse, centred (phase ramps instead of (-1)^n for odd N) / uncentred; two batch elements."""
    u = field(N, 11000 + N, 2, dtype)
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.fft2d(d, direction, centered)
    want = np.stack([oracle.fft2d(u[b], direction, centered) for b in range(2)])
    assert_parity(d.cpu().numpy(), want, dtype)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", SIZES)
def test_propagate_as_and_direct_any_n(torch_cuda, B, oracle, N, dtype):
    """Angular spectrum (FFT-order frequencies of an odd grid) and direct Fresnel with z > 0 and z < 0, per-batch
    wavelength and pitch."""
    u = field(N, 11100 + N, 2, dtype)
    dx, lam = np.array([1e-5, 1.3e-5]), np.array([1e-6, 0.7e-6])
    zc = N * dx[0] ** 2 / lam[0]
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.propagate_as(d, dx, lam, 0.3 * zc)
    want = oracle.propagate_as_batch(u, dx, lam, 0.3 * zc)
    assert_parity(d.cpu().numpy(), want, dtype)
    for z in (1.4 * zc, -0.9 * zc):
        d = to_dev(torch_cuda, u, dtype)
        px = plan.propagate_direct(d, dx, lam, z)
        w = []
        for b in range(2):
            f, dxo = oracle.propagate_direct(u[b], dx[b], lam[b], z)
            assert px[b] == pytest.approx(dxo, rel=1e-15)
            w.append(f)
        assert_parity(d.cpu().numpy(), np.stack(w), dtype, f"direct z={z:.3g}")


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", [175, 335, 360, 700, 1025])
def test_surface_and_train_any_n(torch_cuda, B, oracle, N, dtype):
    """The fused surface (lens + amplitude + OPD + angular spectrum), the stand-alone operators, the broadband image
    and a train with AUTO (a mix of angular spectrum and direct) on non-power-of-two grids."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    u = field(N, 11200 + N, 2, dtype)
    dx, lam = np.array([2e-5, 2e-5]), np.array([0.9e-6, 0.8e-6])
    zc = N * dx[0] ** 2 / lam[0]
    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, 2e-5, 3.0, 15e-9, 11201)
    da, do = map_dev(torch_cuda, amp, dtype), map_dev(torch_cuda, opd, dtype)
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.surface_as(d, dx, lam, 0.8, da, do, 0.25 * zc)
    want = oracle.surface_as_batch(u, dx, lam, 0.8, map_host(amp, dtype), map_host(opd, dtype), 0.25 * zc)
    assert_parity(d.cpu().numpy(), want, dtype)
    # stand-alone operators
    d = to_dev(torch_cuda, u, dtype)
    plan.apply_qpf(d, dx, lam, -0.5)
    plan.apply_mask(d, da, do, lam)
    want = np.stack([oracle.apply_mask(oracle.apply_qpf(u[b], dx[b], lam[b], -0.5), map_host(amp, dtype), map_host(opd, dtype), lam[b])
                     for b in range(2)])
    assert_parity(d.cpu().numpy(), want, dtype)
    # broadband image of an odd number of pixels
    img = map_dev(torch_cuda, np.zeros((N, N)), dtype)
    plan.accumulate_intensity(d, [0.4, 0.6], img)
    wimg = oracle.broadband_image(want, [0.4, 0.6])
    got = img.cpu().numpy().astype(np.float64)
    assert np.linalg.norm(got - wimg) / np.linalg.norm(wimg) <= (1e-11 if dtype == "c128" else 2e-5)
    # train, AUTO rule
    surfs = [Surface(0.6, 0.4 * zc, amp, opd), Surface(-0.9, 1.7 * zc, None, opd), Surface(math.inf, 0.0, amp, None),
             Surface(0.8, 0.3 * zc)]
    maps = [(map_dev(torch_cuda, s.amp, dtype), map_dev(torch_cuda, s.opd, dtype)) for s in surfs]
    d = to_dev(torch_cuda, u, dtype)
    px, used = plan.system_run(d, dx, lam, surfs, maps=maps)
    assert used[:3] == [0, 1, -1]
    got = d.cpu().numpy().reshape(2, N, N)
    hs = [Surface(s.f, s.z, map_host(s.amp, dtype), map_host(s.opd, dtype)) for s in surfs]
    for b in range(2):
        w, dxo, used_o = oracle.system_run(u[b], dx[b], lam[b], hs)
        assert used_o == used and px[b] == pytest.approx(dxo, rel=1e-14)
        assert_parity(got[b][None], w[None], dtype, f"train, wavelength {b}")


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_n2800_the_papers_size(torch_cuda, B, oracle, dtype):
    """N = 2800 = 2^4 5^2 7: one angular-spectrum step of a config-4 style random field and one
    direct step, whole field against the oracle's O(N^3) DFT (tens of seconds of host time)."""
    N = 2800
    u = field(N, 11300, 1, dtype)
    dx, lam = np.array([1e-5]), np.array([1e-6])
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.propagate_as(d, dx, lam, 0.1)
    want = oracle.propagate_as(u[0], dx[0], lam[0], 0.1)
    assert_parity(d.cpu().numpy(), want[None], dtype)
    d = to_dev(torch_cuda, u, dtype)
    px = plan.propagate_direct(d, dx, lam, 0.5)
    want, dxo = oracle.propagate_direct(u[0], dx[0], lam[0], 0.5)
    assert px[0] == pytest.approx(dxo, rel=1e-15)
    assert_parity(d.cpu().numpy(), want[None], dtype)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", [1400, 1500, 2400])
def test_register_resident_all_modes(torch_cuda, B, oracle, N, dtype):
    """N = 1400 = 5 * 5 * 7 * 8, 1500 = 3 * 5 * 5 * 5 * 4 and 2400 = 3 * 5 * 5 * 2 * 16 (five stages) on the register-resident
    mixed-radix pass (mr_kernel.cuh): inverse and centred transforms, direct Fresnel with z < 0, and a surface with both maps
    on the load of the row pass."""
    from paper_1806_06467_b200 import inputs
    u = field(N, 11500, 1, dtype)
    dx, lam = np.array([1.5e-5]), np.array([0.8e-6])
    zc = N * dx[0] ** 2 / lam[0]
    plan = B.Plan(N, 1, dtype)
    for direction, centered in ((-1, False), (+1, True)):
        d = to_dev(torch_cuda, u, dtype)
        plan.fft2d(d, direction, centered)
        assert_parity(d.cpu().numpy(), oracle.fft2d(u[0], direction, centered)[None], dtype, f"fft2d {direction} {centered}")
    d = to_dev(torch_cuda, u, dtype)
    px = plan.propagate_direct(d, dx, lam, -1.2 * zc)
    want, dxo = oracle.propagate_direct(u[0], dx[0], lam[0], -1.2 * zc)
    assert px[0] == pytest.approx(dxo, rel=1e-15)
    assert_parity(d.cpu().numpy(), want[None], dtype, "direct z < 0")
    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, 1.5e-5, 3.0, 15e-9, 11501)
    d = to_dev(torch_cuda, u, dtype)
    plan.surface_as(d, dx, lam, 0.7, map_dev(torch_cuda, amp, dtype), map_dev(torch_cuda, opd, dtype), 0.2 * zc)
    want = oracle.surface_as_batch(u, dx, lam, 0.7, map_host(amp, dtype), map_host(opd, dtype), 0.2 * zc)
    assert_parity(d.cpu().numpy(), want, dtype, "surface")


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_n4100_the_papers_appendix_b_grid(torch_cuda, B, oracle, dtype):
    """N = 4100 = 41 * 4 * 5 * 5: `WFIRSTSPC(npix=1025)` at beam ratio 0.25.  The oracle's O(N^3)
    transform takes minutes at this size, so: (a) the centred forward transform on a 15 x 15 subset of its outputs, each
    computed one by one by the oracle's matrix Fourier transform (pinned to the centred FFT by P24 / P24b); (b) the inverse
    transform undoes it; (c) angular spectrum at half the Talbot distance of a field with a 100-pixel period: the exact
    half-period shift (P6), which fails for any error in the transfer function's frequency index."""
    N = 4100
    u = field(N, 11600, 1, dtype)
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.fft2d(d, +1, True)
    got = d.cpu().numpy()[0]
    lam, f, dx = 1e-6, 1.0, 1e-5
    nb, stride = 15, 257
    v = oracle.mft(u[0], dx, nb, stride * lam * f / (N * dx), lam, f, +1) / (dx * dx / (1j * lam * f))
    idx = N // 2 + (np.arange(nb) - nb // 2) * stride
    scale = np.linalg.norm(got) / N                      # rms of the whole spectrum: the bar is relative to the field, not the subset
    assert np.linalg.norm(got[np.ix_(idx, idx)] - v) / (nb * scale) <= TOL[dtype]
    assert np.abs(got[np.ix_(idx, idx)] - v).max() <= 50 * TOL[dtype] * np.abs(got).max()
    assert np.linalg.norm(got) == pytest.approx(N * np.linalg.norm(u[0]), rel=10 * TOL[dtype])   # Parseval
    plan.fft2d(d, -1, True)
    assert_parity(d.cpu().numpy(), u, dtype, "inverse of forward")
    # Talbot: period 100 px, z_T = 2 d^2 / lambda; at z_T / 2 the field comes back shifted by half a period along both axes
    per = 100
    cell = field(per, 11601, 1, dtype)[0]
    w = np.tile(cell, (N // per, N // per))[None]
    dxs, lams = np.array([1e-5]), np.array([1e-6])
    zt = 2 * (per * dxs[0]) ** 2 / lams[0]
    d = to_dev(torch_cuda, w, dtype)
    plan.propagate_as(d, dxs, lams, zt / 2)
    assert_parity(d.cpu().numpy(), np.roll(w, (per // 2, per // 2), axis=(1, 2)), dtype, "half Talbot distance")


MR_SIZES = [700, 1000, 1200, 1400, 1500, 2000, 2400, 2800, 3000, 3600, 4000, 5000, 5600, 6000]


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", MR_SIZES)
def test_register_resident_pass_equals_the_shared_memory_pass(torch_cuda, B, N, dtype):
    """Cross-check (not the parity proof: that is the oracle at 700 ... 2800 above): at EVERY size of the register-resident
    pass the results equal those of the shared-memory mixed-radix pass (FRESNEL_NO_MR=1 at plan creation), which the oracle
    covers at many sizes -- angular spectrum, an inverse centred transform and direct Fresnel, to rounding."""
    import os
    u = field(N, 11700 + N, 1, dtype)
    dx, lam = np.array([1.1e-5]), np.array([0.9e-6])
    zc = N * dx[0] ** 2 / lam[0]
    out = {}
    for tag in ("fast", "shared"):
        if tag == "shared":
            os.environ["FRESNEL_NO_MR"] = "1"
        try:
            plan = B.Plan(N, 1, dtype)
        finally:
            os.environ.pop("FRESNEL_NO_MR", None)
        res = []
        d = to_dev(torch_cuda, u, dtype); plan.propagate_as(d, dx, lam, 0.3 * zc); res.append(d.cpu().numpy())
        d = to_dev(torch_cuda, u, dtype); plan.fft2d(d, -1, True); res.append(d.cpu().numpy())
        d = to_dev(torch_cuda, u, dtype); plan.propagate_direct(d, dx, lam, 1.3 * zc); res.append(d.cpu().numpy())
        out[tag] = res
        plan.close()
    tol = 1e-13 if dtype == "c128" else 2e-6
    for a, b, what in zip(out["fast"], out["shared"], ("angular spectrum", "inverse centred transform", "direct Fresnel")):
        assert np.linalg.norm(a - b) / np.linalg.norm(b) <= tol, f"N = {N} {what}"


def test_n1100_radix_11_and_capacity_limits(torch_cuda, B, oracle):
    """1100 = 2^2 5^2 11 exercises the radix-11 butterfly; sizes beyond the shared-memory capacity are refused."""
    import ctypes
    N = 1100
    u = field(N, 11400, 1, "c128")
    plan = B.Plan(N, 1, "c128")
    d = to_dev(torch_cuda, u, "c128")
    plan.fft2d(d, +1, False)
    assert_parity(d.cpu().numpy(), oracle.fft2d(u[0], +1, False)[None], "c128")
    h = ctypes.c_void_p()
    assert B.lib().fresnel_plan_create(ctypes.byref(h), 4268, 1, 1) == 2       # 2^2 11 97: Bluestein would need M >= 8535
    assert B.lib().fresnel_plan_create(ctypes.byref(h), 7300, 1, 1) == 2
