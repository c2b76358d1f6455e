"""Gaussian pilot-beam trains on the GPU (fresnel_system_run_pilot; PAPER.md:29,
:228-259), run with -m gpu.  The stored array, the pixel pitch, the pilot state and the legs taken must equal the
oracle's (oracle.system_run_pilot, pinned by P20-P23 against the Gaussian-beam closed forms) on the same inputs.
"""
import math

import numpy as np
import pytest

from test_gpu_parity import TOL, assert_parity, field, map_dev, map_host, to_dev

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


def same_state(got, want):
    for g, w in zip(got, want):
        if math.isinf(w):
            assert math.isinf(g)
        else:
            assert g == pytest.approx(w, rel=1e-13, abs=1e-300)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_pilot_free_space_gaussian(torch_cuda, B, oracle, dtype):
    """P20 on the GPU: from the waist to 0.3 zR (PTP), to 8 zR (WTS, spherical reference) and back (STW)."""
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam, w0 = 512, 1e-5, 1e-6, 2e-4
    zR = math.pi * w0 * w0 / lam
    x = (np.arange(N) - N // 2) * dx
    u0 = np.exp(-(x[None, :] ** 2 + x[:, None] ** 2) / w0 ** 2).astype(np.complex128)[None]
    if dtype == "c64":
        u0 = u0.astype(np.complex64).astype(np.complex128)
    plan = B.Plan(N, 1, dtype)
    for z, legs_want in ((0.3 * zR, [(1, 0)]), (8.0 * zR, [(0, 2)])):
        d = to_dev(torch_cuda, u0, dtype)
        px, st, legs = plan.system_run_pilot(d, [dx], [lam], [Surface(math.inf, z)], w0)
        want, dxo, st_o, legs_o = oracle.system_run_pilot(u0[0], dx, lam, [Surface(math.inf, z)], w0)
        assert legs == legs_o == legs_want and px[0] == pytest.approx(dxo, rel=1e-15)
        same_state(st[0], st_o)
        assert_parity(d.cpu().numpy(), want[None], dtype)
    # back to the waist from 8 zR
    px2, st2, legs2 = plan.system_run_pilot(d, px, [lam], [Surface(math.inf, -8.0 * zR)], w0, state=st)
    back, dx2, st2_o, legs2_o = oracle.system_run_pilot(want, dxo, lam, [Surface(math.inf, -8.0 * zR)], w0, state=st_o)
    assert legs2 == legs2_o == [(3, 0)] and px2[0] == pytest.approx(dx2, rel=1e-14)
    same_state(st2[0], st2_o)
    assert_parity(d.cpu().numpy(), back[None], dtype)
    assert np.linalg.norm(d.cpu().numpy().reshape(N, N) - u0[0]) / np.linalg.norm(u0[0]) <= (1e-10 if dtype == "c128" else 1e-4)


def test_pilot_config2_through_lenses(torch_cuda, B, oracle):
    """Config 2 (1024^2 complex128 Gaussian, three lenses) under the pilot-beam rule: stored field, pitch, state and
    legs after every surface against the oracle, which lands on the ABCD closed form (P22)."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    w0 = 2e-3
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    o, dxo, st_o = wl.field[0], float(wl.dx[0]), None
    px, st = wl.dx.copy(), None
    for i, s in enumerate(wl.surfaces):
        px, st, legs = plan.system_run_pilot(d, px, wl.lam, [s], w0, state=st)
        o, dxo, st_o, legs_o = oracle.system_run_pilot(o, dxo, wl.lam[0], [s], w0, state=st_o)
        assert legs == legs_o, f"surface {i}"
        assert px[0] == pytest.approx(dxo, rel=1e-14)
        same_state(st[0], st_o)
        assert_parity(d.cpu().numpy(), o[None], "c128", f"surface {i}")
    # the whole train in one call gives the same
    d2 = to_dev(torch_cuda, wl.field, "c128")
    px2, st2, legs2 = plan.system_run_pilot(d2, wl.dx, wl.lam, wl.surfaces, w0)
    assert px2[0] == pytest.approx(px[0], rel=1e-15)
    assert_parity(d2.cpu().numpy(), o[None], "c128")


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_pilot_coronagraph_shaped_train_with_masks_and_batch(torch_cuda, B, oracle, dtype):
    """The shape of the paper's App. B prescription: pupil -> lens -> focal-plane mask -> lens ->
    Lyot-plane mask -> lens -> image, every lens with a surface-error map; two wavelengths that take the same legs."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    N, dx = 512, 2e-5
    lam = np.array([0.60e-6, 0.62e-6])
    R = 2.0e-3                                            # pupil radius = pilot beam radius
    pupil = inputs.circular_aperture(N, R / dx)
    occ = (inputs.centred_r2_px(N) > 6 ** 2).astype(np.float64)
    lyot = inputs.circular_aperture(N, 0.8 * R / dx)
    opd = [inputs.psd_map(N, dx, 3.0, 8e-9, 12000 + i) for i in range(3)]
    f = 0.4
    surfs = [Surface(math.inf, 0.05, pupil, None), Surface(f, f, None, opd[0]), Surface(math.inf, f, occ, None),
             Surface(f, 0.1, lyot, opd[1]), Surface(f, f, None, opd[2])]
    u = np.ones((2, N, N), dtype=np.complex128)
    plan = B.Plan(N, 2, dtype)
    maps = [(map_dev(torch_cuda, s.amp, dtype), map_dev(torch_cuda, s.opd, dtype)) for s in surfs]
    d = to_dev(torch_cuda, u, dtype)
    px, st, legs = plan.system_run_pilot(d, [dx, dx], lam, surfs, R, maps=maps)
    got = d.cpu().numpy().reshape(2, N, N)
    hs = [Surface(s.f, s.z, map_host(s.amp, dtype), map_host(s.opd, dtype)) for s in surfs]
    kinds = set()
    for b in range(2):
        want, dxo, st_o, legs_o = oracle.system_run_pilot(u[b], dx, lam[b], hs, R)
        assert legs == legs_o
        kinds |= {l for pair in legs_o for l in pair}
        assert px[b] == pytest.approx(dxo, rel=1e-13)
        same_state(st[b], st_o)
        assert_parity(got[b][None], want[None], dtype, f"wavelength {b}")
    assert {1, 2, 3} <= kinds                            # the train exercises PTP, WTS and STW


def test_pilot_errors_enqueue_nothing(torch_cuda, B):
    from paper_1806_06467_b200.inputs import Surface
    N = 256
    plan = B.Plan(N, 2, "c128")
    u = field(N, 12100, 2)
    d = to_dev(torch_cuda, u, "c128")
    l0 = plan.launch_count()
    w0 = 3e-4                                             # zR = 0.47 m at 0.6 um, 0.28 m at 1 um
    with pytest.raises(B.FresnelError) as e:              # 0.35 m: inside the Rayleigh range of one wavelength only
        plan.system_run_pilot(d, [1e-5, 1e-5], [0.6e-6, 1.0e-6], [Surface(math.inf, 0.35)], w0)
    assert e.value.status == 2
    with pytest.raises(B.FresnelError) as e:
        plan.system_run_pilot(d, [1e-5, 1e-5], [0.6e-6, 0.6e-6], [Surface(math.inf, 0.1), Surface(0.0, 0.1)], w0)
    assert e.value.status == 1
    with pytest.raises(B.FresnelError):
        plan.system_run_pilot(d, [1e-5, 1e-5], [0.6e-6, 0.6e-6], [Surface(math.inf, 0.1)], -1.0)
    assert plan.launch_count() == l0
    assert np.array_equal(d.cpu().numpy().reshape(u.shape), u)
