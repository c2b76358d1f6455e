"""GPU-vs-oracle parity (run with -m gpu on a B200).  Every call goes through the C ABI of
libfresnel.so (paper_1806_06467_b200.binding); the expected values come from oracle/ on the same
seeded inputs.  Bar (BASELINE.json:north_star): relative L2 per batch element, max over the batch,
<= 1e-11 for complex128 and <= 2e-5 for complex64.  For c64 the inputs are rounded to float32
first and the oracle runs in double on those rounded values.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-11, "c64": 2e-5}
ALL_N = [64, 128, 256, 512, 1024, 2048]


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B(torch_cuda):
    from paper_1806_06467_b200 import binding
    binding.lib()          # fails loudly if libfresnel.so is missing
    return binding


def rel_batch(got, want):
    """Relative L2 per batch element, max over the batch (the north-star metric, reading g20) -- and, beside it,
    a bound on the LARGEST pointwise deviation, max|g-o| <= 50 * tol * max|o| (asserted whenever the caller's
    tolerance is one of the two north-star ones), so that a defect confined to a few lines of a large grid cannot
    hide in the norm.  Returns the L2 figure; the max-abs figure of the last call is kept in rel_batch.last_max."""
    got = np.asarray(got).reshape(want.shape)
    errs, mx = [], []
    for b in range(want.shape[0]):
        d = got[b] - want[b]
        errs.append(np.linalg.norm(d) / np.linalg.norm(want[b]))
        mx.append(np.abs(d).max() / np.abs(want[b]).max())
    rel_batch.last_max = float(max(mx))
    return float(max(errs))


rel_batch.last_max = 0.0


def assert_parity(got, want, dtype, what=""):
    """The parity bar: relative L2 <= tol AND max|g-o| <= 50*tol*max|o| (per batch element)."""
    e = rel_batch(got, want)
    assert e <= TOL[dtype], f"{what}: relative L2 {e:.3e} > {TOL[dtype]:.0e}"
    assert rel_batch.last_max <= 50 * TOL[dtype], f"{what}: max-abs {rel_batch.last_max:.3e} > {50 * TOL[dtype]:.0e} of max|o|"


def field(N, seed, batch=1, dtype="c128"):
    from paper_1806_06467_b200 import inputs
    u = inputs.random_field(N, seed, batch)
    if dtype == "c64":
        u = u.astype(np.complex64).astype(np.complex128)
    return u


def to_dev(torch, u, dtype):
    t = torch.from_numpy(np.ascontiguousarray(u))
    if dtype == "c64":
        t = t.to(torch.complex64)
    return t.cuda().contiguous()


def map_dev(torch, m, dtype):
    if m is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(m))
    return (t.to(torch.float32) if dtype == "c64" else t).cuda().contiguous()


def map_host(m, dtype):
    """what the GPU sees: for c64 the maps are float32"""
    if m is None:
        return None
    return m.astype(np.float32).astype(np.float64) if dtype == "c64" else m


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", ALL_N)
@pytest.mark.parametrize("direction,centered", [(+1, False), (-1, False), (+1, True), (-1, True)])
def test_fft2d(torch_cuda, B, oracle, N, dtype, direction, centered):
    u = field(N, 100 + N, 2, dtype)
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.fft2d(d, direction, centered)
    want = np.stack([oracle.fft2d(u[b], direction, centered) for b in range(2)])
    assert_parity(d.cpu().numpy(), want, dtype)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", ALL_N)
def test_propagate_as(torch_cuda, B, oracle, N, dtype):
    """config-4 style: random field, lambda 1e-6, z 0.5, dx 1e-5; two batch elements with different
    wavelength and pitch so that per-batch tables are exercised."""
    u = field(N, 4000 + int(math.log2(N)), 2, dtype)
    dx, lam, z = np.array([1e-5, 1.3e-5]), np.array([1e-6, 0.7e-6]), 0.5
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.propagate_as(d, dx, lam, z)
    want = oracle.propagate_as_batch(u, dx, lam, z)
    assert_parity(d.cpu().numpy(), want, dtype)
    # negative z undoes it (g10)
    plan.propagate_as(d, dx, lam, -z)
    assert rel_batch(d.cpu().numpy(), u) <= 4 * TOL[dtype]


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", [64, 256, 1024, 2048])
@pytest.mark.parametrize("z", [0.7, -0.4])
def test_propagate_direct(torch_cuda, B, oracle, N, dtype, z):
    u = field(N, 200 + N, 2, dtype)
    dx, lam = np.array([2e-5, 1.5e-5]), np.array([1e-6, 0.633e-6])
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    dx_out = plan.propagate_direct(d, dx, lam, z)
    want = []
    for b in range(2):
        w, dxo = oracle.propagate_direct(u[b], dx[b], lam[b], z)
        assert dx_out[b] == pytest.approx(dxo, rel=1e-15)
        want.append(w)
    assert_parity(d.cpu().numpy(), np.stack(want), dtype)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", [64, 512, 2048])
def test_apply_qpf_and_mask(torch_cuda, B, oracle, N, dtype):
    from paper_1806_06467_b200 import inputs
    u = field(N, 300 + N, 2, dtype)
    dx, lam, f = np.array([2e-5, 1e-5]), np.array([550e-9, 600e-9]), 0.2     # corner phase ~ 1e3..2e4 rad
    plan = B.Plan(N, 2, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.apply_qpf(d, dx, lam, -f)
    want = np.stack([oracle.apply_qpf(u[b], dx[b], lam[b], -f) for b in range(2)])
    assert_parity(d.cpu().numpy(), want, dtype)

    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, 2e-5, 3.0, 20e-9, 77)
    for a, o in [(amp, opd), (None, opd), (amp, None)]:
        d = to_dev(torch_cuda, u, dtype)
        plan.apply_mask(d, map_dev(torch_cuda, a, dtype), map_dev(torch_cuda, o, dtype), lam)
        want = np.stack([oracle.apply_mask(u[b], map_host(a, dtype), map_host(o, dtype), lam[b]) for b in range(2)])
        assert_parity(d.cpu().numpy(), want, dtype)
    # both NULL: no-op
    d = to_dev(torch_cuda, u, dtype)
    plan.apply_mask(d, None, None, lam)
    assert rel_batch(d.cpu().numpy(), u) <= (1e-7 if dtype == "c64" else 0.0)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", [128, 1024, 2048])
def test_surface_as_fused_vs_oracle_and_primitives(torch_cuda, B, oracle, N, dtype):
    from paper_1806_06467_b200 import inputs
    u = field(N, 500 + N, 2, dtype)
    dx, lam, f, z = np.array([2e-5, 2e-5]), np.array([550e-9, 640e-9]), 0.8, 0.35
    amp = inputs.circular_aperture(N, N / 4)
    opd = inputs.psd_map(N, 2e-5, 3.0, 10e-9, 78)
    plan = B.Plan(N, 2, dtype)
    da, do = map_dev(torch_cuda, amp, dtype), map_dev(torch_cuda, opd, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.surface_as(d, dx, lam, f, da, do, z)
    want = oracle.surface_as_batch(u, dx, lam, f, map_host(amp, dtype), map_host(opd, dtype), z)
    assert_parity(d.cpu().numpy(), want, dtype)
    # fused == primitives chained, to rounding
    e = to_dev(torch_cuda, u, dtype)
    plan.apply_qpf(e, dx, lam, -f)
    plan.apply_mask(e, da, do, lam)
    plan.propagate_as(e, dx, lam, z)
    assert rel_batch(e.cpu().numpy(), d.cpu().numpy().reshape(2, N, N)) <= TOL[dtype]
    # z == 0: optic only
    g = to_dev(torch_cuda, u, dtype)
    plan.surface_as(g, dx, lam, f, da, do, 0.0)
    want0 = np.stack([oracle.apply_mask(oracle.apply_qpf(u[b], dx[b], lam[b], -f), map_host(amp, dtype),
                                        map_host(opd, dtype), lam[b]) for b in range(2)])
    assert_parity(g.cpu().numpy(), want0, dtype)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_mask_large_opd_both_phasor_branches(torch_cuda, B, oracle, dtype):
    """Eq. 3 with an OPD of several waves: the kernel's small-phase polynomial (|OPD/lambda| <= 1/8) and
    its library branch are both taken, stand-alone and fused into the row pass."""
    from paper_1806_06467_b200 import inputs
    N = 512
    u = field(N, 911, 1, dtype)
    lam, dx = np.array([600e-9]), np.array([1e-5])
    opd = inputs.psd_map(N, 1e-5, 2.5, 400e-9, 912)             # RMS 2/3 wave: |u| spans 0 .. ~3 turns
    assert (np.abs(opd / lam[0]) > 0.125).mean() > 0.3 and (np.abs(opd / lam[0]) <= 0.125).mean() > 0.05
    plan = B.Plan(N, 1, dtype)
    do = map_dev(torch_cuda, opd, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.apply_mask(d, None, do, lam)
    want = oracle.apply_mask(u[0], None, map_host(opd, dtype), lam[0])[None]
    assert_parity(d.cpu().numpy(), want, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.surface_as(d, dx, lam, None, None, do, 0.02)
    want = oracle.surface_as_batch(u, dx, lam, None, None, map_host(opd, dtype), 0.02)
    assert_parity(d.cpu().numpy(), want, dtype)


@pytest.mark.parametrize("dtype,N,batch", [("c128", 256, 3), ("c64", 512, 2), ("c128", 1024, 1), ("c64", 128, 70)])
def test_accumulate_intensity(torch_cuda, B, oracle, dtype, N, batch):
    """Broadband image (NEXT-3): image += sum_b w_b |U_b|^2 against the oracle, on top of a
    non-zero image, batch both below and above the 64 weights one launch carries."""
    u = field(N, 1300 + N, batch, dtype)
    w = np.random.Generator(np.random.PCG64(N)).uniform(0.1, 2.0, batch)
    img0 = np.random.Generator(np.random.PCG64(N + 1)).uniform(0.0, 1.0, (N, N))
    plan = B.Plan(N, batch, dtype)
    d = to_dev(torch_cuda, u, dtype)
    img = map_dev(torch_cuda, img0, dtype)
    plan.accumulate_intensity(d, w, img)
    want = map_host(img0, dtype).copy()
    for b in range(batch):
        want = oracle.accumulate_intensity(u[b], w[b], want)
    got = img.cpu().numpy().astype(np.float64)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) <= (1e-14 if dtype == "c128" else 1e-6)
    # the wavefront is read only
    assert rel_batch(d.cpu().numpy(), u) <= (1e-7 if dtype == "c64" else 0.0)


def test_config1(torch_cuda, B, oracle):
    from paper_1806_06467_b200 import inputs
    wl = inputs.config1()
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    plan.propagate_as(d, wl.dx, wl.lam, wl.surfaces[0].z)
    want = oracle.propagate_as_batch(wl.field, wl.dx, wl.lam, wl.surfaces[0].z)
    assert_parity(d.cpu().numpy(), want, "c128")


def test_config2_both_variants(torch_cuda, B, oracle):
    """Gaussian-beam chain: GPU vs oracle after every stage, AS and direct variants."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    lam = wl.lam
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    o = wl.field[0]
    for s in wl.surfaces:
        plan.surface_as(d, wl.dx, lam, s.f, None, None, s.z)
        o = oracle.surface_as(o, wl.dx[0], lam[0], s.f, None, None, s.z)
        assert_parity(d.cpu().numpy(), o[None], "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    o, dx_o, dx_g = wl.field[0], float(wl.dx[0]), wl.dx.copy()
    for s in wl.surfaces:
        plan.apply_qpf(d, dx_g, lam, -s.f)
        dx_g = plan.propagate_direct(d, dx_g, lam, s.z)
        o = oracle.apply_qpf(o, dx_o, lam[0], -s.f)
        o, dx_o = oracle.propagate_direct(o, dx_o, lam[0], s.z)
        assert dx_g[0] == pytest.approx(dx_o, rel=1e-15)
        assert_parity(d.cpu().numpy(), o[None], "c128")


def test_config3_reduced_chain(torch_cuda, B, oracle):
    """Shaped-pupil-coronagraph analog at N=512 (full recipe, scaled masks), all 20 surfaces."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config3(N=512)
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    o = wl.field[0]
    for i, s in enumerate(wl.surfaces):
        plan.surface_as(d, wl.dx, wl.lam, s.f, map_dev(torch_cuda, s.amp, "c128"), map_dev(torch_cuda, s.opd, "c128"), s.z)
        o = oracle.surface_as(o, wl.dx[0], wl.lam[0], s.f, s.amp, s.opd, s.z)
        if i in (0, 6, 12, 19):
            assert_parity(d.cpu().numpy(), o[None], "c128", f"surface {i}")


def test_config3_full_size_bench_step(torch_cuda, B, oracle):
    """The step bench.py times: config 3 at its full size (N=2048, complex128, 20 surfaces with their maps), same
    call sequence, whole field against the oracle at the end of the chain and at three surfaces on the way."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config3()
    assert wl.N == 2048 and len(wl.surfaces) == 20
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    maps = [(map_dev(torch_cuda, s.amp, "c128"), map_dev(torch_cuda, s.opd, "c128")) for s in wl.surfaces]
    o = wl.field[0]
    for i, s in enumerate(wl.surfaces):
        plan.surface_as(d, wl.dx, wl.lam, s.f, maps[i][0], maps[i][1], s.z)
        o = oracle.surface_as(o, wl.dx[0], wl.lam[0], s.f, s.amp, s.opd, s.z)
        if i in (0, 6, 12, 19):
            assert_parity(d.cpu().numpy(), o[None], "c128", f"surface {i}")


def test_config5_full_size_all_wavelengths(torch_cuda, B, oracle):
    """Config 5 at full size (16 wavelengths x 4096^2 complex64, 10 planes, one call per plane for the whole batch,
    the launch configuration bench.py --workload cfg5 times): EVERY wavelength's whole field against the oracle
    after plane 10 (160 oracle surface-propagations), plus the invariant the chain has -- lenses and propagation are
    unitary, so each wavelength's energy after the pupil mask of plane 0 is conserved."""
    torch = torch_cuda
    from paper_1806_06467_b200 import inputs
    wl = inputs.config5()
    assert wl.N == 4096 and wl.batch == 16 and len(wl.surfaces) == 10
    plan = B.Plan(wl.N, wl.batch, "c64")
    d = to_dev(torch, wl.field, "c64")
    maps = [(map_dev(torch, s.amp, "c64"), map_dev(torch, s.opd, "c64")) for s in wl.surfaces]
    e_after_pupil = None
    for i, s in enumerate(wl.surfaces):
        plan.surface_as(d, wl.dx, wl.lam, s.f, maps[i][0], maps[i][1], s.z)
        if i == 0:
            e_after_pupil = (d.abs().double() ** 2).sum(dim=(-2, -1)).cpu().numpy()
    e_end = (d.abs().double() ** 2).sum(dim=(-2, -1)).cpu().numpy()
    assert np.all(np.abs(e_end / e_after_pupil - 1) <= 2e-5)
    got = d.cpu().numpy().reshape(wl.batch, wl.N, wl.N)
    del d
    for b in range(wl.batch):
        o = wl.field[b].astype(np.complex64).astype(np.complex128)
        for s in wl.surfaces:
            o = oracle.surface_as(o, wl.dx[b], wl.lam[b], s.f, map_host(s.amp, "c64"), map_host(s.opd, "c64"), s.z)
        assert_parity(got[b][None], o[None], "c64", f"wavelength {b}")


def test_config5_reduced_batch(torch_cuda, B, oracle):
    """Polychromatic batch at N=512, 4 wavelengths, 10 planes, c64."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config5(N=512, batch=4)
    plan = B.Plan(wl.N, wl.batch, "c64")
    d = to_dev(torch_cuda, wl.field, "c64")
    o = wl.field.copy()
    for s in wl.surfaces:
        plan.surface_as(d, wl.dx, wl.lam, s.f, map_dev(torch_cuda, s.amp, "c64"), map_dev(torch_cuda, s.opd, "c64"), s.z)
        o = oracle.surface_as_batch(o, wl.dx, wl.lam, s.f, map_host(s.amp, "c64"), map_host(s.opd, "c64"), s.z)
    assert_parity(d.cpu().numpy(), o, "c64")


@pytest.mark.parametrize("dtype,N", [("c128", 4096), ("c64", 4096), ("c64", 8192), ("c128", 8192)])
def test_large_grids_sampled(torch_cuda, B, oracle, dtype, N):
    """Full bench sizes: the oracle's radix-2 FFT still finishes in seconds at 4096/8192, so compare
    the whole field for one AS step of config 4."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config4(N, dtype)
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, wl.field, dtype)
    plan.propagate_as(d, wl.dx, wl.lam, wl.surfaces[0].z)
    want = oracle.propagate_as_batch(wl.field, wl.dx, wl.lam, wl.surfaces[0].z)
    assert_parity(d.cpu().numpy(), want, dtype)


@pytest.mark.parametrize("dtype,N", [("c128", 4096), ("c64", 8192)])
def test_large_grids_fused_surface_and_direct(torch_cuda, B, oracle, dtype, N):
    """Large grids through the fused surface (lens + amplitude + OPD + AS: phasor and chirps on the row pass,
    per-row factor on its store) and through direct Fresnel with z < 0, whole field against the oracle."""
    from paper_1806_06467_b200 import inputs
    u = field(N, 2000 + N, 1, dtype)
    dx, lam = np.array([1e-5]), np.array([633e-9])
    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, 1e-5, 2.5, 15e-9, 2001)
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.surface_as(d, dx, lam, 1.3, map_dev(torch_cuda, amp, dtype), map_dev(torch_cuda, opd, dtype), 0.2)
    want = oracle.surface_as(u[0], dx[0], lam[0], 1.3, map_host(amp, dtype), map_host(opd, dtype), 0.2)
    assert_parity(d.cpu().numpy(), want[None], dtype)
    px = plan.propagate_direct(d, dx, lam, -0.9)
    want, dxo = oracle.propagate_direct(want, dx[0], lam[0], -0.9)
    assert px[0] == pytest.approx(dxo, rel=1e-15)
    assert_parity(d.cpu().numpy(), want[None], dtype)


LARGE = [("c128", 4096), ("c64", 4096), ("c128", 8192), ("c64", 8192)]


@pytest.mark.parametrize("dtype,N", LARGE)
@pytest.mark.parametrize("direction,centered", [(+1, False), (-1, False), (+1, True), (-1, True)])
def test_fft2d_large_grids(torch_cuda, B, oracle, N, dtype, direction, centered):
    """fresnel_fft2d at the sweep's large sizes (own template instantiations: 4096 = 16*16*16, 8192 = 16*16*16*2,
    own tile geometry): forward / inverse x centred / uncentred, whole field against the oracle's literal
    ifftshift -> radix-2 fft2 -> fftshift (PAPER.md:47 "significantly larger arrays", :79, :121-125)."""
    u = field(N, 7000 + N, 1, dtype)
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.fft2d(d, direction, centered)
    want = oracle.fft2d(u[0], direction, centered)[None]
    assert_parity(d.cpu().numpy(), want, dtype)


@pytest.mark.parametrize("dtype,N", LARGE)
@pytest.mark.parametrize("z", [1.1, -0.6])
def test_propagate_direct_large_grids(torch_cuda, B, oracle, N, dtype, z):
    """Direct Fresnel with z > 0 (forward kernel) and z < 0 (inverse kernel) at N = 4096 / 8192, both precisions
    (PAPER.md:29, 53)."""
    u = field(N, 7100 + N, 1, dtype)
    dx, lam = np.array([1.5e-5]), np.array([0.8e-6])
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, u, dtype)
    px = plan.propagate_direct(d, dx, lam, z)
    want, dxo = oracle.propagate_direct(u[0], dx[0], lam[0], z)
    assert px[0] == pytest.approx(dxo, rel=1e-15)
    assert_parity(d.cpu().numpy(), want[None], dtype)


@pytest.mark.parametrize("dtype,N", LARGE)
def test_apply_qpf_and_mask_large_grids(torch_cuda, B, oracle, N, dtype):
    """The stand-alone one-pass operators (Eq. 2, Eq. 3) at N = 4096 / 8192: corner phases of 1e4..1e5 rad."""
    from paper_1806_06467_b200 import inputs
    u = field(N, 7200 + N, 1, dtype)
    dx, lam, f = np.array([1e-5]), np.array([600e-9]), 0.35
    plan = B.Plan(N, 1, dtype)
    d = to_dev(torch_cuda, u, dtype)
    plan.apply_qpf(d, dx, lam, -f)
    want = oracle.apply_qpf(u[0], dx[0], lam[0], -f)
    assert_parity(d.cpu().numpy(), want[None], dtype)
    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, 1e-5, 3.0, 20e-9, 7201)
    d = to_dev(torch_cuda, u, dtype)
    plan.apply_mask(d, map_dev(torch_cuda, amp, dtype), map_dev(torch_cuda, opd, dtype), lam)
    want = oracle.apply_mask(u[0], map_host(amp, dtype), map_host(opd, dtype), lam[0])
    assert_parity(d.cpu().numpy(), want[None], dtype)


def test_config3_second_run_auto_mixes_as_and_direct(torch_cuda, B, oracle):
    """SURVEY.md sec. 8(d) cfg3 "second run": the same 20 surfaces at full size (N=2048, complex128) through
    fresnel_system_run with method AUTO -- direct Fresnel wherever z_s >= N dx^2 / lambda of the CURRENT pixel
    pitch (z_c = 1.49 m at the start), angular spectrum elsewhere.  Whole field against the oracle's train."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config3()
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    maps = [(map_dev(torch_cuda, s.amp, "c128"), map_dev(torch_cuda, s.opd, "c128")) for s in wl.surfaces]
    px, used = plan.system_run(d, wl.dx, wl.lam, wl.surfaces, maps=maps)
    want, dxo, used_o = oracle.system_run(wl.field[0], wl.dx[0], wl.lam[0], wl.surfaces)
    assert used == used_o
    assert 0 in used and 1 in used, f"expected a mix of angular spectrum and direct, got {used}"
    assert px[0] == pytest.approx(dxo, rel=1e-13)
    assert_parity(d.cpu().numpy(), want[None], "c128")


def test_error_codes(torch_cuda, B):
    import ctypes
    L = B.lib()
    h = ctypes.c_void_p()
    assert L.fresnel_plan_create(ctypes.byref(h), 7919, 1, 1) == 2          # UNSUPPORTED: a prime above the Bluestein capacity
    assert L.fresnel_plan_create(ctypes.byref(h), 7300, 1, 1) == 2          # smooth, but two line buffers exceed shared memory
    assert L.fresnel_plan_create(ctypes.byref(h), 32, 1, 1) == 2
    assert L.fresnel_plan_create(ctypes.byref(h), 256, 0, 1) == 1           # INVALID_ARG
    assert L.fresnel_plan_create(None, 256, 1, 1) == 1
    plan = B.Plan(256, 1, "c128")
    d = torch_cuda.zeros(256, 256, dtype=torch_cuda.complex128, device="cuda")
    with pytest.raises(B.FresnelError):
        plan.apply_qpf(d, [1e-5], [1e-6], 0.0)
    with pytest.raises(B.FresnelError):
        plan.propagate_direct(d, [1e-5], [1e-6], 0.0)
    with pytest.raises(B.FresnelError):
        plan.propagate_as(d, [1e-5], [-1e-6], 0.1)
    with pytest.raises(B.FresnelError):
        plan.propagate_as(d, [0.0], [1e-6], 0.1)
    with pytest.raises(B.FresnelError):
        plan.propagate_as(d, [1e-5], [1e-6], float("nan"))
    with pytest.raises(B.FresnelError):
        plan.fft2d(d, 0, False)
    with pytest.raises(B.FresnelError):
        plan.surface_as(d, [1e-5], [1e-6], 0.0, None, None, 0.1)
    # z = 0 AS is the identity and launches nothing
    n0 = plan.launch_count()
    plan.propagate_as(d, [1e-5], [1e-6], 0.0)
    assert plan.launch_count() == n0
    assert L.fresnel_plan_destroy(None) == 0


def test_cuda_graph_capture_of_a_chain(torch_cuda, B, oracle):
    """Hot calls enqueue only (no allocation, no sync): a chain can be captured and replayed."""
    torch = torch_cuda
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    s = torch.cuda.Stream()
    plan = B.Plan(wl.N, 1, "c128", stream=s)
    d = to_dev(torch, wl.field, "c128")
    src = d.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        for surf in wl.surfaces:                       # warm-up outside capture
            plan.surface_as(d, wl.dx, wl.lam, surf.f, None, None, surf.z)
        s.synchronize()
        d.copy_(src)
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            for surf in wl.surfaces:
                plan.surface_as(d, wl.dx, wl.lam, surf.f, None, None, surf.z)
    d.copy_(src)
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    o = wl.field[0]
    for surf in wl.surfaces:
        o = oracle.surface_as(o, wl.dx[0], wl.lam[0], surf.f, None, None, surf.z)
    assert_parity(d.cpu().numpy(), o[None], "c128")


# ---- train of surfaces (NEXT-1 reduced, reading g13b) ---------------------------------------------
def test_system_run_config2_auto_takes_direct_and_matches_oracle(torch_cuda, B, oracle):
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    px, used = plan.system_run(d, wl.dx, wl.lam, wl.surfaces)
    want, dxo, used_o = oracle.system_run(wl.field[0], wl.dx[0], wl.lam[0], wl.surfaces)
    assert used == used_o == [1, 1, 1]
    assert px[0] == pytest.approx(dxo, rel=1e-15)
    assert_parity(d.cpu().numpy(), want[None], "c128")
    # forced angular spectrum: the surface_as chain
    d = to_dev(torch_cuda, wl.field, "c128")
    px, used = plan.system_run(d, wl.dx, wl.lam, wl.surfaces, methods=[B.METHOD_AS] * 3)
    want, _, _ = oracle.system_run(wl.field[0], wl.dx[0], wl.lam[0], wl.surfaces, methods=[0, 0, 0])
    assert used == [0, 0, 0] and px[0] == wl.dx[0]
    assert_parity(d.cpu().numpy(), want[None], "c128")


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_system_run_mixed_train_with_masks_and_batch(torch_cuda, B, oracle, dtype):
    """Lens + maps + AS below z_c, optic only at z = 0, lens merged into the direct transform above z_c (also
    with a mask on that surface and with z < 0), two wavelengths on the same side of their z_c."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    N = 512
    dx, lam = np.array([2e-5, 2e-5]), np.array([1.0e-6, 0.9e-6])
    zc = N * dx[0] ** 2 / lam[0]                                    # 0.2048 m (0.2276 m for the second wavelength)
    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, 2e-5, 3.0, 15e-9, 41)
    surfs = [Surface(0.6, 0.4 * zc, amp, opd), Surface(math.inf, 0.0, None, opd), Surface(-0.9, 1.7 * zc, amp, opd),
             Surface(0.8, -1.3 * 1.7 ** 2 * zc), Surface(math.inf, 0.3 * zc)]
    u = field(N, 77, 2, dtype)
    plan = B.Plan(N, 2, dtype)
    maps = [(map_dev(torch_cuda, s.amp, dtype), map_dev(torch_cuda, s.opd, dtype)) for s in surfs]
    d = to_dev(torch_cuda, u, dtype)
    px, used = plan.system_run(d, dx, lam, surfs, maps=maps)
    assert used == [0, -1, 1, 1, 0]
    got = d.cpu().numpy().reshape(2, N, N)
    for b in range(2):
        hs = [Surface(s.f, s.z, map_host(s.amp, dtype), map_host(s.opd, dtype)) for s in surfs]
        want, dxo, used_o = oracle.system_run(u[b], dx[b], lam[b], hs)
        assert used_o == used
        assert px[b] == pytest.approx(dxo, rel=1e-14)
        assert_parity(got[b][None], want[None], dtype)


def test_system_run_errors_enqueue_nothing(torch_cuda, B):
    from paper_1806_06467_b200.inputs import Surface
    N = 256
    plan = B.Plan(N, 2, "c128")
    u = field(N, 5, 2)
    d = to_dev(torch_cuda, u, "c128")
    l0 = plan.launch_count()
    dx, lam = np.array([1e-5, 1e-5]), np.array([0.5e-6, 1.0e-6])     # z_c = 0.0512 and 0.0256 m
    with pytest.raises(B.FresnelError) as e:                         # the batch straddles z_c
        plan.system_run(d, dx, lam, [Surface(math.inf, 0.01), Surface(math.inf, 0.04)])
    assert e.value.status == 2
    with pytest.raises(B.FresnelError) as e:                         # bad focal length in the LAST surface
        plan.system_run(d, dx, lam, [Surface(math.inf, 0.01), Surface(0.0, 0.01)])
    assert e.value.status == 1
    assert plan.launch_count() == l0                                 # validated before anything was enqueued
    assert rel_batch(d.cpu().numpy(), u) == 0.0
    # forcing the method resolves the straddle
    plan.system_run(d, dx, lam, [Surface(math.inf, 0.04)], methods=[B.METHOD_AS])


def test_system_run_as_one_cuda_graph(torch_cuda, B, oracle):
    torch = torch_cuda
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    s = torch.cuda.Stream()
    plan = B.Plan(wl.N, 1, "c128", stream=s)
    d = to_dev(torch, wl.field, "c128")
    src = d.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        plan.system_run(d, wl.dx, wl.lam, wl.surfaces)              # warm-up outside capture
        s.synchronize()
        d.copy_(src)
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            plan.system_run(d, wl.dx, wl.lam, wl.surfaces)
    d.copy_(src)
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    want, _, _ = oracle.system_run(wl.field[0], wl.dx[0], wl.lam[0], wl.surfaces)
    assert_parity(d.cpu().numpy(), want[None], "c128")


def test_table_cache_eviction_long_train(torch_cuda, B, oracle):
    """40 surfaces with distinct lenses and distances need 80 chirp tables, more than the plan caches (64): the
    least-recently-used slots are rebuilt in stream order.  Run the train twice (second time with a partly stale
    cache) against the oracle."""
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam = 128, np.array([2e-5]), np.array([0.8e-6])
    r = np.random.Generator(np.random.PCG64(404))
    surfs = [Surface(float(r.uniform(0.3, 2.0)), float(r.uniform(0.002, 0.02))) for _ in range(40)]
    u = field(N, 405, 1)
    plan = B.Plan(N, 1, "c128")
    want, _, _ = oracle.system_run(u[0], dx[0], lam[0], surfs, methods=[0] * 40)
    for _ in range(2):
        d = to_dev(torch_cuda, u, "c128")
        px, used = plan.system_run(d, dx, lam, surfs, methods=[B.METHOD_AS] * 40)
        assert used == [0] * 40 and px[0] == dx[0]
        assert_parity(d.cpu().numpy(), want[None], "c128")
