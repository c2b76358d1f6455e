"""Pins for the CPU oracle (DESIGN.md "Oracle pins" P0..P13): closed forms, exact identities, brute
force and the paper's own worked example.  Nothing here touches the GPU or the CUDA library.

Each pin is chosen so that a plausible mistake in oracle/fresnel_oracle.c (a dropped term, a wrong
sign or index, a transposed operand, a wrong scale) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
from scipy.special import j1

HERE = os.path.dirname(os.path.abspath(__file__))
PI_L = 4 * np.arctan(np.longdouble(1))      # pi to long-double precision (np.pi is only a double)


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def rnd(N, seed):
    r = np.random.Generator(np.random.PCG64(seed))
    return r.standard_normal((N, N)) + 1j * r.standard_normal((N, N))


def coords(N, dx):
    c = (np.arange(N) - N // 2) * dx
    return c[None, :], c[:, None]     # x (varies along k, the fast axis), y (along j)


# ---------------------------------------------------------------- P0 / definition of the DFT itself
def test_dft2_naive_closed_forms(oracle):
    """The brute-force DFT against closed forms: a delta transforms to a constant, a single complex
    exponential exp(+2 pi i (j p0 + k q0)/N) transforms (forward kernel exp(-...)) to N^2 at
    [p0, q0] -- pins sign, axis order and scaling of the definition everything else rests on."""
    N = 16
    d = np.zeros((N, N), complex)
    d[0, 0] = 1.0
    assert np.allclose(oracle.dft2_naive(d, -1), 1.0, atol=1e-15)
    p0, q0 = 3, 5
    j, k = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    e = np.exp(2j * np.pi * (j * p0 + k * q0) / N)
    F = oracle.dft2_naive(e, -1)
    expect = np.zeros((N, N), complex)
    expect[p0, q0] = N * N
    assert np.abs(F - expect).max() < 1e-11
    # inverse kernel: same input lands at [-p0, -q0] with scale 1/N^2 ... and e itself maps from a delta
    G = oracle.dft2_naive(expect, +1)
    assert np.abs(G - e).max() < 1e-13
    # a shifted delta gives the conjugate-phase ramp: F[p,q] = exp(-2 pi i (p j0 + q k0)/N)
    d = np.zeros((N, N), complex)
    d[2, 7] = 1.0
    F = oracle.dft2_naive(d, -1)
    assert np.abs(F - np.exp(-2j * np.pi * (j * 2 + k * 7) / N)).max() < 1e-14


@pytest.mark.parametrize("N", [8, 16, 32, 64])
@pytest.mark.parametrize("sign", [-1, +1])
def test_P0_fft2_vs_bruteforce(oracle, N, sign):
    u = rnd(N, 10 + N)
    assert rel(oracle.fft2(u, sign), oracle.dft2_naive(u, sign)) <= 1e-13


def test_fft2_reduces_to_library_routine(oracle):
    u = rnd(512, 77)
    assert rel(oracle.fft2(u, -1), np.fft.fft2(u)) <= 1e-14
    assert rel(oracle.fft2(u, +1), np.fft.ifft2(u)) <= 1e-14


# ---------------------------------------------------------------- P1 round trip
def test_P1_round_trip(oracle):
    u = rnd(256, 1)
    assert rel(oracle.fft2(oracle.fft2(u, -1), +1), u) <= 1e-14
    assert rel(oracle.fft2d(oracle.fft2d(u, oracle.FORWARD, 1), oracle.INVERSE, 1), u) <= 1e-14


# ---------------------------------------------------------------- P2 inverse pairs
def test_P2_inverse_pairs(oracle):
    N, dx, lam, z = 1024, 2e-5, 1e-6, 0.7
    u = rnd(N, 2)
    assert rel(oracle.propagate_as(oracle.propagate_as(u, dx, lam, z), dx, lam, -z), u) <= 1e-13
    assert rel(oracle.apply_qpf(oracle.apply_qpf(u, dx, lam, z), dx, lam, -z), u) <= 1e-14
    v, dx1 = oracle.propagate_direct(u, dx, lam, z)
    assert dx1 == pytest.approx(lam * z / (N * dx), rel=1e-15)
    w, dx2 = oracle.propagate_direct(v, dx1, lam, -z)
    assert dx2 == pytest.approx(dx, rel=1e-14)
    # dx2 equals dx only to one rounding (dx1 is a rounded double); the ~1e3 rad corner phase of the
    # last chirp turns that 1e-16 relative pitch error into ~1e-13 of field error.
    assert rel(w, u) <= 1e-12


# ---------------------------------------------------------------- P3 Parseval
def test_P3_parseval(oracle):
    N, dx, lam, z = 512, 2e-5, 0.8e-6, 0.3
    u = rnd(N, 3)
    e0 = np.sum(np.abs(u) ** 2)
    v = oracle.propagate_as(u, dx, lam, z)
    assert np.sum(np.abs(v) ** 2) / e0 == pytest.approx(1.0, abs=1e-13)
    w, dx1 = oracle.propagate_direct(u, dx, lam, z)
    assert np.sum(np.abs(w) ** 2) * dx1 ** 2 / (e0 * dx ** 2) == pytest.approx(1.0, abs=1e-13)
    F = oracle.fft2(u, -1)
    assert np.sum(np.abs(F) ** 2) / (N * N * e0) == pytest.approx(1.0, abs=1e-13)


# ---------------------------------------------------------------- P4 Gaussian beam closed form
def gaussian_closed_form(N, dx, lam, w0, z):
    """U(r, z) = (q0/q) exp(i pi r^2/(lam q)), q0 = -i zR, q = q0 + z, zR = pi w0^2/lam
    (textbook Gaussian beam: w(z) = w0 sqrt(1+(z/zR)^2), on-axis amplitude w0/w, Gouy phase
    -atan(z/zR), curvature R = z (1+(zR/z)^2)); no piston exp(ikz) (reading g5)."""
    x, y = coords(N, dx)
    zR = math.pi * w0 * w0 / lam
    q0 = -1j * zR
    q = q0 + z
    return (q0 / q) * np.exp(1j * np.pi * (x * x + y * y) / (lam * q))


def test_P4_gaussian_beam_as(oracle):
    N, dx, lam, w0 = 1024, 2e-5, 1.064e-6, 2e-3
    u0 = gaussian_closed_form(N, dx, lam, w0, 0.0)
    assert np.abs(u0.imag).max() < 1e-15 and u0[N // 2, N // 2].real == pytest.approx(1.0)
    for z, tol in [(0.5, 1e-9), (2.0, 1e-9), (5.0, 1e-8)]:
        v = oracle.propagate_as(u0, dx, lam, z)
        assert rel(v, gaussian_closed_form(N, dx, lam, w0, z)) <= tol
    # the physics the north star names: w(z) = w0 sqrt(1 + (z/zR)^2) from the second moment
    z = 5.0
    v = oracle.propagate_as(u0, dx, lam, z)
    x, y = coords(N, dx)
    I = np.abs(v) ** 2
    w_num = math.sqrt(2.0 * np.sum(I * (x * x + y * y)) / np.sum(I))
    zR = math.pi * w0 * w0 / lam
    assert w_num == pytest.approx(w0 * math.sqrt(1 + (z / zR) ** 2), rel=1e-6)
    assert abs(v[N // 2, N // 2]) == pytest.approx(1 / math.sqrt(1 + (z / zR) ** 2), rel=1e-9)
    assert np.angle(v[N // 2, N // 2]) == pytest.approx(-math.atan(z / zR), abs=1e-9)


@pytest.mark.parametrize("z", [0.5, 2.0, 5.0, -0.5])
def test_P4_gaussian_beam_direct(oracle, z):
    N, dx, lam, w0 = 1024, 2e-5, 1.064e-6, 2e-3
    u0 = gaussian_closed_form(N, dx, lam, w0, 0.0)
    v, dx1 = oracle.propagate_direct(u0, dx, lam, z)
    assert dx1 == pytest.approx(lam * abs(z) / (N * dx), rel=1e-15)
    if z == 0.5:
        assert dx1 == pytest.approx(2.598e-5, rel=2e-4)
    assert rel(v, gaussian_closed_form(N, dx1, lam, w0, z)) <= 1e-9


# ---------------------------------------------------------------- P5 Gaussian through lenses (config 2)
def abcd_chain(lam, w0, steps):
    """Complex beam parameter through thin lenses and free space:
    lens: 1/q <- 1/q - 1/f;  free space z: A <- A q/(q+z), q <- q+z;  field A exp(i pi r^2/(lam q))."""
    q = -1j * math.pi * w0 * w0 / lam
    A = 1.0 + 0j
    out = []
    for f, z in steps:
        q = 1.0 / (1.0 / q - 1.0 / f)
        A = A * q / (q + z)
        q = q + z
        out.append((q, A))
    return out


def test_P5_gaussian_lens_chain(oracle):
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    N, dx, lam, w0 = wl.N, float(wl.dx[0]), float(wl.lam[0]), 2e-3
    steps = [(s.f, s.z) for s in wl.surfaces]
    ref = abcd_chain(lam, w0, steps)
    # beam parameters after each stage (values recorded in SURVEY.md sec. 8(c) P5)
    w = [math.sqrt(lam / (math.pi * (1 / q).imag)) for q, _ in ref]
    assert w[0] == pytest.approx(84.67e-6, rel=1e-3)
    assert w[1] == pytest.approx(3.0003e-3, rel=1e-4)
    assert w[2] == pytest.approx(4.0036e-3, rel=1e-4)
    assert [abs(A) for _, A in ref] == pytest.approx([23.621, 0.6666, 0.49955], rel=2e-4)

    # direct chain: pixel scale changes at every step
    u, d = wl.field[0], dx
    tol_direct = [1e-8, 1e-8, 1e-8]
    for (f, z), (q, A), tol in zip(steps, ref, tol_direct):
        u = oracle.apply_qpf(u, d, lam, -f)
        u, d = oracle.propagate_direct(u, d, lam, z)
        x, y = coords(N, d)
        assert rel(u, A * np.exp(1j * np.pi * (x * x + y * y) / (lam * q))) <= tol
        I = np.abs(u) ** 2
        w_num = math.sqrt(2.0 * np.sum(I * (x * x + y * y)) / np.sum(I))
        assert w_num == pytest.approx(math.sqrt(lam / (math.pi * (1 / q).imag)), rel=1e-5)
    assert d == pytest.approx(3.464e-5, rel=2e-4)

    # angular-spectrum chain: fixed pixel scale; the beam reaches the grid edge at stages 2 and 3
    # (half-width/w = 3.4 then 2.6), so those tolerances are grid truncation, not oracle error.
    u = wl.field[0]
    x, y = coords(N, dx)
    for (f, z), (q, A), tol in zip(steps, ref, [1e-9, 1e-4, 5e-3]):
        u = oracle.surface_as(u, dx, lam, f, None, None, z)
        assert rel(u, A * np.exp(1j * np.pi * (x * x + y * y) / (lam * q))) <= tol


# ---------------------------------------------------------------- P6 Talbot, exact
def test_P6_talbot_exact(oracle):
    N, dx, lam, dpx = 256, 1e-5, 1e-6, 16
    cell = rnd(dpx, 6)
    u = np.tile(cell, (N // dpx, N // dpx))
    d = dpx * dx
    zT = 2 * d * d / lam
    assert rel(oracle.propagate_as(u, dx, lam, zT), u) <= 1e-13
    half = oracle.propagate_as(u, dx, lam, zT / 2)
    assert rel(half, np.roll(u, (dpx // 2, dpx // 2), axis=(0, 1))) <= 1e-13
    assert rel(half, u) > 0.5      # and it is NOT the unshifted field


# ---------------------------------------------------------------- P7 Talbot, the paper's example
def read_golden(name):
    out = {}
    with open(os.path.join(HERE, "golden", name)) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


def test_P7_talbot_paper_example(oracle):
    g = read_golden("talbot_paper_example.txt")
    lam = 1e-6                                             # reading g14
    D, cyc, amp_m = g["aperture_diameter_m"], g["cycles_per_aperture"], g["wfe_amplitude_m"]
    d = D / cyc                                            # grating period: 1 mm
    ZT = 2 * (D / cyc) ** 2 / lam                          # Eq. 1
    assert d == pytest.approx(1e-3) and ZT == pytest.approx(2.0)
    N, dx = 256, d / 16
    x, _ = coords(N, dx)
    eps = 2 * math.pi * amp_m / lam
    c = np.cos(2 * np.pi * x / d) * np.ones((N, 1))
    u0 = np.exp(1j * eps * c)
    # complete phase -> amplitude conversion at 0.25 Z_T
    u = oracle.propagate_as(u0, dx, lam, g["full_conversion_zt"] * ZT)
    a = np.abs(u)
    coef = np.sum((a - a.mean()) * c) / np.sum(c * c) / eps
    assert coef == pytest.approx(1.0, abs=5e-4)           # +eps*cos: the opposite sign of H gives -1
    assert np.abs(a - (1 + eps * c)).max() <= 0.75 * eps * eps
    ph = np.angle(u)
    assert np.sqrt(np.mean((ph - ph.mean()) ** 2)) <= 1e-12   # phase is flat
    # partial conversion at 0.05 Z_T: amplitude modulation eps*sin(2 pi z/Z_T), residual phase eps*cos(2 pi z/Z_T)
    zf = g["partial_conversion_zt"]
    u = oracle.propagate_as(u0, dx, lam, zf * ZT)
    a = np.abs(u)
    coef = np.sum((a - a.mean()) * c) / np.sum(c * c) / eps
    assert coef == pytest.approx(math.sin(2 * math.pi * zf), abs=2e-3)
    ph = np.angle(u)
    pcoef = np.sum((ph - ph.mean()) * c) / np.sum(c * c) / eps
    assert pcoef == pytest.approx(math.cos(2 * math.pi * zf), abs=2e-3)


# ---------------------------------------------------------------- P8 Airy far field
def test_P8_airy(oracle):
    from paper_1806_06467_b200 import inputs
    N, dx, lam, apx, f = 1024, 1e-5, 1e-6, 32, 0.5
    ap = inputs.circular_aperture(N, apx).astype(complex)
    u = oracle.apply_qpf(ap, dx, lam, -f)
    v, dx1 = oracle.propagate_direct(u, dx, lam, f)
    centre = v[N // 2, N // 2]
    expect_centre = ap.sum().real * dx * dx / (1j * lam * f)
    assert abs(centre - expect_centre) <= 1e-12 * abs(expect_centre)
    assert centre.imag == pytest.approx(-0.6418, abs=2e-4) and abs(centre.real) < 1e-12
    a = apx * dx
    rp = (np.arange(N) - N // 2) * dx1
    sl = slice(N // 2 - 60, N // 2 + 61)
    vv = 2 * np.pi * a * np.abs(rp[sl]) / (lam * f)
    with np.errstate(invalid="ignore", divide="ignore"):
        airy = np.where(vv == 0, 1.0, 2 * j1(vv) / vv)
    model = (np.pi * a * a / (lam * f)) * np.abs(airy)
    peak = model.max()
    assert np.abs(np.abs(v[N // 2, sl]) - model).max() <= 5e-3 * peak      # row cut
    assert np.abs(np.abs(v[sl, N // 2]) - model).max() <= 5e-3 * peak      # column cut
    prof = np.abs(v[N // 2, N // 2:N // 2 + 40])
    first_min = int(np.argmax((prof[1:-1] < prof[:-2]) & (prof[1:-1] < prof[2:]))) + 1
    assert abs(first_min - 0.6098 * N * dx / a) <= 1.0                      # 19.51 px predicted


# ---------------------------------------------------------------- P9 AS == direct at the critical distance
def test_P9_as_equals_direct_at_critical_distance(oracle):
    N, dx, lam = 1024, 2e-5, 1e-6
    zc = N * dx * dx / lam
    x, y = coords(N, dx)
    u = np.exp(-(x * x + y * y) / (2e-3) ** 2) * np.exp(0.1j * np.cos(2 * np.pi * x / (32 * dx)))
    a = oracle.propagate_as(u, dx, lam, zc)
    b, dx1 = oracle.propagate_direct(u, dx, lam, zc)
    assert dx1 == pytest.approx(dx, rel=1e-14)
    assert rel(a, b) <= 1e-12


# ---------------------------------------------------------------- P10 semigroup
def test_P10_semigroup(oracle):
    N, dx, lam = 256, 1e-5, 1e-6
    u = rnd(N, 10)
    a = oracle.propagate_as(oracle.propagate_as(u, dx, lam, 0.013), dx, lam, 0.021)
    assert rel(a, oracle.propagate_as(u, dx, lam, 0.034)) <= 1e-13
    assert rel(oracle.propagate_as(u, dx, lam, 0.0), u) <= 1e-14          # z = 0 is the identity (g11)


# ---------------------------------------------------------------- P11 shift bookkeeping
def test_P11_shift_bookkeeping(oracle):
    N, dx, lam, z = 256, 1e-5, 1e-6, 0.02
    u = rnd(N, 11)
    # literal shifted AS == unshifted AS with H in FFT order (same long-double phase evaluation)
    m = np.where(np.arange(N) < N // 2, np.arange(N), np.arange(N) - N).astype(np.longdouble)
    fq = m / (np.longdouble(N) * np.longdouble(dx))
    th = -PI_L * np.longdouble(lam) * np.longdouble(z) * (fq[None, :] ** 2 + fq[:, None] ** 2)
    H = np.cos(th).astype(np.float64) + 1j * np.sin(th).astype(np.float64)
    unshifted = oracle.fft2(oracle.fft2(u, -1) * H, +1)
    assert rel(unshifted, oracle.propagate_as(u, dx, lam, z)) <= 1e-15
    # the rotations themselves
    assert np.array_equal(oracle.fftshift(u), np.fft.fftshift(u))
    assert np.array_equal(oracle.ifftshift(u), np.fft.ifftshift(u))
    # centred FFT == s * fft2(s * u), s = (-1)^(j+k): exactly
    j, k = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    s = (-1.0) ** (j + k)
    assert np.array_equal(oracle.fft2d(u, oracle.FORWARD, 1), s * oracle.fft2(s * u, -1))
    assert np.array_equal(oracle.fft2d(u, oracle.INVERSE, 1), s * oracle.fft2(s * u, +1))


# ---------------------------------------------------------------- P12 QPF structure
def test_P12_qpf_structure(oracle):
    N, dx, lam, z = 512, 2e-5, 550e-9, -0.2          # lens f = 0.2 m: corner phase ~ 1.5e3 rad
    Q = oracle.apply_qpf(np.ones((N, N), complex), dx, lam, z)
    assert Q[N // 2, N // 2] == 1.0 + 0j
    assert np.array_equal(Q[1:, :], Q[:0:-1, :]) and np.array_equal(Q[:, 1:], Q[:, :0:-1])
    assert np.array_equal(Q, Q.T)
    assert np.abs(np.abs(Q) - 1).max() < 1e-15
    c = ((np.arange(N) - N // 2) * np.longdouble(dx))
    th = PI_L * c * c / (np.longdouble(lam) * np.longdouble(z))
    t = np.cos(th).astype(np.float64) + 1j * np.sin(th).astype(np.float64)
    assert np.abs(Q - t[:, None] * t[None, :]).max() <= 1e-14
    # sign and scale of the phase (reading g1): one pixel off axis the phase is pi dx^2/(lam z)
    assert np.angle(Q[N // 2, N // 2 + 1]) == pytest.approx(math.pi * dx * dx / (lam * z), rel=1e-12)
    # x runs along the fast axis, y along the slow one; the chirp is the same in both
    assert Q[N // 2 + 3, N // 2] == Q[N // 2, N // 2 + 3]


# ---------------------------------------------------------------- P13 mask special cases
def test_P13_mask_special_cases(oracle):
    N, lam = 128, 633e-9
    u = rnd(N, 13)
    assert np.array_equal(oracle.apply_mask(u, None, None, lam), u)
    assert np.array_equal(oracle.apply_mask(u, np.ones((N, N)), np.zeros((N, N)), lam), u)
    assert rel(oracle.apply_mask(u, None, np.full((N, N), lam), lam), u) <= 1e-15
    A = (np.random.Generator(np.random.PCG64(5)).random((N, N)) < 0.5).astype(float)
    v = oracle.apply_mask(u, A, None, lam)
    assert np.all(v[A == 0] == 0) and np.array_equal(v[A == 1], u[A == 1])
    # quarter-wave OPD multiplies by +i (sign of Eq. 3, reading g3)
    w = oracle.apply_mask(u, None, np.full((N, N), lam / 4), lam)
    assert rel(w, 1j * u) <= 1e-15
    # non-uniform map, against the definition evaluated with numpy
    opd = np.random.Generator(np.random.PCG64(6)).normal(0, 20e-9, (N, N))
    assert rel(oracle.apply_mask(u, A, opd, lam), u * A * np.exp(2j * np.pi * opd / lam)) <= 1e-15


def test_surface_as_is_the_literal_composition(oracle):
    N, dx, lam = 256, 2e-5, 550e-9
    u = rnd(N, 14)
    r = np.random.Generator(np.random.PCG64(7))
    A, opd = (r.random((N, N)) < 0.7).astype(float), r.normal(0, 10e-9, (N, N))
    lit = oracle.propagate_as(oracle.apply_mask(oracle.apply_qpf(u, dx, lam, -0.8), A, opd, lam), dx, lam, 0.4)
    assert np.array_equal(oracle.surface_as(u, dx, lam, 0.8, A, opd, 0.4), lit)
    assert np.array_equal(oracle.surface_as(u, dx, lam, math.inf, None, None, 0.4), oracle.propagate_as(u, dx, lam, 0.4))


def test_oracle_rejects_bad_arguments(oracle):
    u = rnd(64, 15)
    with pytest.raises(oracle.OracleError):
        oracle.apply_qpf(u, 1e-5, 1e-6, 0.0)
    with pytest.raises(oracle.OracleError):
        oracle.propagate_direct(u, 1e-5, 1e-6, 0.0)
    with pytest.raises(oracle.OracleError):
        oracle.propagate_as(u, -1e-5, 1e-6, 0.1)
    with pytest.raises(oracle.OracleError):
        oracle.dft2_naive(rnd(128, 1), -1)


# ---- P14: broadband image ("repeated for all of the wavelengths") ----
def test_p14_accumulate_intensity_closed_forms(oracle):
    N = 64
    img0 = np.full((N, N), 2.0)
    u = np.full((N, N), 3 + 4j)
    assert np.array_equal(oracle.accumulate_intensity(u, 0.5, img0), np.full((N, N), 14.5))      # 2 + 0.5*25, exact
    assert np.array_equal(img0, np.full((N, N), 2.0))                                           # caller's image untouched
    v = rnd(N, 21)
    assert np.array_equal(oracle.accumulate_intensity(v, 0.0, img0), img0)                      # zero weight
    one = oracle.accumulate_intensity(v, 1.0)
    assert rel(one, v.real ** 2 + v.imag ** 2) <= 1e-16
    assert rel(oracle.accumulate_intensity(v, 0.25, one), 1.25 * one) <= 1e-15                  # linear in the weight
    # a pure phase factor does not change the image
    assert rel(oracle.accumulate_intensity(v * np.exp(0.7j), 1.0), one) <= 1e-15


def test_p14_broadband_energy_and_gaussian_beam_intensity(oracle):
    """Two wavelengths of the same Gaussian waist: sum_b w_b |U_b|^2 after propagation equals
    sum_b w_b (w0/w_b(z))^2 exp(-2 r^2 / w_b(z)^2), w_b(z) = w0 sqrt(1 + (z/zR_b)^2), and carries the
    weighted input energy (Parseval per wavelength)."""
    N, dx, w0, z = 512, 4e-5, 2e-3, 1.5
    lams, wts = np.array([500e-9, 1000e-9]), np.array([0.3, 0.7])
    x = (np.arange(N) - N // 2) * dx
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    u0 = np.exp(-r2 / w0 ** 2).astype(np.complex128)
    stack = np.stack([oracle.propagate_as(u0, dx, lam, z) for lam in lams])
    img = oracle.broadband_image(stack, wts)
    want = np.zeros((N, N))
    for lam, wt in zip(lams, wts):
        zr = np.pi * w0 ** 2 / lam
        wz = w0 * np.sqrt(1 + (z / zr) ** 2)
        want += wt * (w0 / wz) ** 2 * np.exp(-2 * r2 / wz ** 2)
    assert rel(img, want) <= 1e-9
    assert abs(img.sum() / (wts.sum() * (np.abs(u0) ** 2).sum()) - 1) <= 1e-13


# ---- P15: train of surfaces with the sampling rule for the propagator (NEXT-1 reduced, reading g13b) ----
def test_p15_system_run_auto_rule_and_closed_form(oracle):
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    N, dx, lam, w0 = wl.N, float(wl.dx[0]), float(wl.lam[0]), 2e-3
    # config 2: z_c = N dx^2/lam = 0.385, 0.650, 0.866 m along the chain and z = 0.5, 0.75, 1.0 -> direct every time;
    # the result is the ABCD closed form of the three-lens chain (P5) on the final grid
    u, d, used = oracle.system_run(wl.field[0], dx, lam, wl.surfaces)
    assert used == [1, 1, 1]
    q, A = abcd_chain(lam, w0, [(s.f, s.z) for s in wl.surfaces])[-1]
    assert d == pytest.approx(3.464e-5, rel=2e-4)
    x, y = coords(N, d)
    assert rel(u, A * np.exp(1j * np.pi * (x * x + y * y) / (lam * q))) <= 1e-8
    # forced angular spectrum == the surface_as chain, bit for bit; pixel pitch unchanged
    v, dv, used = oracle.system_run(wl.field[0], dx, lam, wl.surfaces, methods=[0, 0, 0])
    w = wl.field[0]
    for s in wl.surfaces:
        w = oracle.surface_as(w, dx, lam, s.f, None, None, s.z)
    assert used == [0, 0, 0] and dv == dx and np.array_equal(v, w)


def test_p15_system_run_threshold_masks_and_zero_distance(oracle):
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam = 128, 2e-5, 1e-6
    zc = N * dx * dx / lam                                            # 0.0512 m
    r = np.random.Generator(np.random.PCG64(31))
    amp, opd = (r.random((N, N)) < 0.8).astype(float), r.normal(0, 15e-9, (N, N))
    u0 = rnd(N, 32)
    surfs = [Surface(0.3, 0.5 * zc, amp, opd), Surface(math.inf, 0.0, None, opd), Surface(-0.7, 1.5 * zc), Surface(math.inf, -0.25 * zc)]
    u, d, used = oracle.system_run(u0, dx, lam, surfs)
    assert used[:3] == [0, -1, 1]                                     # below z_c: AS; z = 0: none; above: direct
    d2 = lam * 1.5 * zc / (N * dx)
    assert d == pytest.approx(d2, rel=1e-15)
    assert used[3] == 0                                               # new pitch 1.5 dx -> z_c grows to 2.25 z_c
    # the literal composition
    w = oracle.propagate_as(oracle.apply_mask(oracle.apply_qpf(u0, dx, lam, -0.3), amp, opd, lam), dx, lam, 0.5 * zc)
    w = oracle.apply_mask(w, None, opd, lam)
    w, dw = oracle.propagate_direct(oracle.apply_qpf(w, dx, lam, 0.7), dx, lam, 1.5 * zc)
    w = oracle.propagate_as(w, dw, lam, -0.25 * zc)
    assert np.array_equal(u, w)
    # from z_c on the rule takes the direct transform, and at z_c the two operators coincide (P9)
    zc1 = zc * (1 + 1e-12)
    a, da, ua = oracle.system_run(u0, dx, lam, [Surface(math.inf, zc1)])
    b, db, ub = oracle.system_run(u0, dx, lam, [Surface(math.inf, zc1)], methods=[0])
    assert ua == [1] and ub == [0] and da == pytest.approx(dx, rel=1e-11) and rel(a, b) <= 1e-9
    assert oracle.system_run(u0, dx, lam, [Surface(math.inf, zc * (1 - 1e-12))])[2] == [0]
    with pytest.raises(oracle.OracleError):
        oracle.system_run(u0, dx, lam, [Surface(0.0, 0.1)])


# ---- P16-P19: grids that are not a power of two (SURVEY.md sec. 8(f) NEXT-2; PAPER.md:137, :172 N = 2800; :259) ----
@pytest.mark.parametrize("N", [9, 12, 15, 35])
@pytest.mark.parametrize("sign", [-1, +1])
def test_P16_dft2_any_vs_bruteforce_and_closed_forms(oracle, N, sign):
    """The plain separable O(N^3) DFT against the literal O(N^4) double sum at odd, even and composite N, and
    against closed forms (single exponential -> N^2 at [p0, q0]; shifted delta -> conjugate phase ramp): pins the
    sign, the axis order, the (k p) mod N indexing and the 1/N^2 of the path every non-power-of-two grid takes."""
    u = rnd(N, 160 + N)
    assert rel(oracle.dft2_any(u, sign), oracle.dft2_naive(u, sign)) <= 1e-13
    assert rel(oracle.fft2(u, sign), oracle.dft2_naive(u, sign)) <= 1e-13          # the dispatch of fft2
    j, k = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    p0, q0 = 2, N - 3
    e = np.exp(2j * np.pi * (j * p0 + k * q0) / N)
    F = oracle.dft2_any(e, -1)
    expect = np.zeros((N, N), complex)
    expect[p0, q0] = N * N
    assert np.abs(F - expect).max() < 1e-10
    d = np.zeros((N, N), complex)
    d[1, N - 2] = 1.0
    assert np.abs(oracle.dft2_any(d, -1) - np.exp(-2j * np.pi * (j * 1 + k * (N - 2)) / N)).max() < 1e-13


def test_P16_dft2_any_special_cases(oracle):
    """At a power of two the plain DFT must agree with the radix-2 path (N = 64); at N = 100 and 175 with the
    library routine (numpy's mixed-radix FFT); forward then inverse is the identity (1/N^2)."""
    u = rnd(64, 161)
    assert rel(oracle.dft2_any(u, -1), oracle.fft2(u, -1)) <= 1e-13
    for N in (100, 175):
        u = rnd(N, 162 + N)
        assert rel(oracle.fft2(u, -1), np.fft.fft2(u)) <= 1e-13
        assert rel(oracle.fft2(u, +1), np.fft.ifft2(u)) <= 1e-13
        assert rel(oracle.fft2(oracle.fft2(u, -1), +1), u) <= 1e-13


@pytest.mark.parametrize("N", [9, 35, 100])
def test_P17_shifts_and_centred_transform_any_N(oracle, N):
    """fftshift / ifftshift are different rotations for odd N (by N//2 and by -(N//2)): exact equality with numpy's,
    and the centred transform of the ABI equals numpy's fftshift(fft2(ifftshift(u)))."""
    u = rnd(N, 170 + N)
    assert np.array_equal(oracle.fftshift(u), np.fft.fftshift(u))
    assert np.array_equal(oracle.ifftshift(u), np.fft.ifftshift(u))
    assert np.array_equal(oracle.ifftshift(oracle.fftshift(u)), u)
    assert rel(oracle.fft2d(u, +1, True), np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(u)))) <= 1e-13
    assert rel(oracle.fft2d(u, -1, True), np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(u)))) <= 1e-13


@pytest.mark.parametrize("N", [700, 625])
def test_P18_gaussian_beam_closed_form_any_N(oracle, N):
    """P4 on a 2^2 5^2 7 grid and on an odd 5^4 grid: the sampled Gaussian beam after angular-spectrum and after
    direct propagation equals (q0/q) exp(i pi r^2/(lambda q)).  For odd N this pins the frequency order
    f_q = q/(N dx) for q <= (N-1)/2, (q-N)/(N dx) above (a wrong split moves one frequency from +f to -f-1/(N dx))
    and the grid centre on pixel N//2."""
    dx, lam, w0 = 2e-5, 1.064e-6, 1.2e-3
    u0 = gaussian_closed_form(N, dx, lam, w0, 0.0)
    for z in (0.4, -0.4):
        assert rel(oracle.propagate_as(u0, dx, lam, z), gaussian_closed_form(N, dx, lam, w0, z)) <= 1e-9
    for z in (0.6, -0.6):
        v, dx1 = oracle.propagate_direct(u0, dx, lam, z)
        assert dx1 == pytest.approx(lam * abs(z) / (N * dx), rel=1e-15)
        assert rel(v, gaussian_closed_form(N, dx1, lam, w0, z)) <= 1e-9


def test_P19_exact_identities_any_N(oracle):
    """Exact identities on non-power-of-two grids: Talbot self-imaging (N = 240, period 16 px; also N = 243 = 3^5
    with period 9 px, an odd grid), the semigroup AS(z1) AS(z2) = AS(z1 + z2), AS(z) AS(-z) = id, Parseval for both
    propagators, direct(-z) direct(z) = id, and AS == direct at z_c = N dx^2 / lambda (N = 300; for odd N the discrete
    chirp exp(i pi m^2 / N) is not its own transform -- a Gauss-sum fact -- so that identity is an even-N one)."""
    dx, lam = 1e-5, 1e-6
    for N, d in ((240, 16), (243, 9)):
        j, k = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
        u = np.exp(1j * 0.3 * np.cos(2 * np.pi * k / d)) * (1 + 0.2 * np.sin(2 * np.pi * j / d))
        zT = 2 * (d * dx) ** 2 / lam
        assert rel(oracle.propagate_as(u, dx, lam, zT), u) <= 1e-12
    N = 300
    u = rnd(N, 190)
    assert rel(oracle.propagate_as(oracle.propagate_as(u, dx, lam, 0.01), dx, lam, 0.02), oracle.propagate_as(u, dx, lam, 0.03)) <= 1e-13
    assert rel(oracle.propagate_as(oracle.propagate_as(u, dx, lam, 0.02), dx, lam, -0.02), u) <= 1e-13
    assert np.sum(np.abs(oracle.propagate_as(u, dx, lam, 0.02)) ** 2) == pytest.approx(np.sum(np.abs(u) ** 2), rel=1e-13)
    v, dx1 = oracle.propagate_direct(u, dx, lam, 0.05)
    assert np.sum(np.abs(v) ** 2) * dx1 ** 2 == pytest.approx(np.sum(np.abs(u) ** 2) * dx ** 2, rel=1e-13)
    w, dx2 = oracle.propagate_direct(v, dx1, lam, -0.05)
    assert dx2 == pytest.approx(dx, rel=1e-15) and rel(w, u) <= 1e-11
    for N in (300,):
        x, y = coords(N, 2e-5)
        g = np.exp(-(x * x + y * y) / (0.8e-3) ** 2) * (1 + 0.05 * np.cos(2 * np.pi * x / 2e-4))
        zc = N * (2e-5) ** 2 / lam
        a = oracle.propagate_as(g, 2e-5, lam, zc)
        b, dxo = oracle.propagate_direct(g, 2e-5, lam, zc)
        assert dxo == pytest.approx(2e-5, rel=1e-14)
        assert rel(a, b) <= 1e-9


# ---- P20-P23: Gaussian pilot-beam propagation (reading g21) ----
def true_field(stored, dx, lam, rref):
    """Put the reference-sphere curvature back: U_true = U_stored exp(i pi r^2/(lam Rref)) (planar: unchanged)."""
    if not math.isfinite(rref):
        return stored
    x, y = coords(stored.shape[0], dx)
    return stored * np.exp(1j * np.pi * (x * x + y * y) / (lam * rref))


def test_P20_pilot_free_space_is_the_gaussian_beam(oracle):
    """The pilot beam IS the Gaussian: start at its waist, go 0.3 zR (stays planar: one PTP leg), 8 zR (one WTS leg,
    spherical reference of radius z) and back.  The TRUE field must equal (q0/q) exp(i pi r^2/(lam q)); the state
    must say w0, waist at 0, position z, Rref = z; on the sphere the stored phase is flat up to the small
    1/R(z) - 1/z mismatch, i.e. far flatter than the true field's."""
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam, w0 = 512, 1e-5, 1e-6, 2e-4
    zR = math.pi * w0 * w0 / lam
    u0 = gaussian_closed_form(N, dx, lam, w0, 0.0)
    v, d1, st, legs = oracle.system_run_pilot(u0, dx, lam, [Surface(math.inf, 0.3 * zR)], w0)
    assert legs == [(oracle.LEG_PTP, 0)] and d1 == dx and st == (w0, 0.0, 0.3 * zR, math.inf)
    assert rel(v, gaussian_closed_form(N, dx, lam, w0, 0.3 * zR)) <= 1e-9
    z = 8.0 * zR
    v, d1, st, legs = oracle.system_run_pilot(u0, dx, lam, [Surface(math.inf, z)], w0)
    assert legs == [(0, oracle.LEG_WTS)]
    assert d1 == pytest.approx(lam * z / (N * dx), rel=1e-15)
    assert st[0] == pytest.approx(w0, rel=1e-15) and st[1] == 0.0 and st[2] == pytest.approx(z) and st[3] == pytest.approx(z)
    assert rel(true_field(v, d1, lam, st[3]), gaussian_closed_form(N, d1, lam, w0, z)) <= 1e-9
    c = N // 2
    w_z = w0 * math.sqrt(1 + (z / zR) ** 2)
    k = int(round(w_z / d1))                                   # one beam radius away from the axis
    stored_dphi = abs(np.angle(v[c, c + k] / v[c, c]))
    true_dphi = math.pi * (k * d1) ** 2 / (lam * z * (1 + (zR / z) ** 2))
    # residual pi w^2/lam (1/R - 1/z) = 65/8 * (1 - 64/65) = 0.125 rad at one beam radius, against 8 rad of true curvature
    assert stored_dphi == pytest.approx(0.125, rel=0.1) and true_dphi > 7.5     # the curvature lives in the reference, not on the grid
    # and back to the waist: one STW leg, the input returns
    w, d2, st2, legs = oracle.system_run_pilot(v, d1, lam, [Surface(math.inf, -z)], w0, state=st)
    assert legs == [(oracle.LEG_STW, 0)] and d2 == pytest.approx(dx, rel=1e-14) and not math.isfinite(st2[3])
    assert rel(w, u0) <= 1e-10


def test_P21_pilot_legs_equal_the_existing_propagators(oracle):
    """Where they coincide the pilot-beam legs ARE the existing operators: inside the Rayleigh range the result is
    propagate_as bit for bit (and two such steps equal one: PTP o PTP = PTP); a waist-to-sphere leg times the output
    chirp is propagate_direct; a sphere-to-waist leg applied to a de-chirped field is propagate_direct too; crossing
    the waist region from sphere to sphere takes STW then WTS and equals direct o direct on the true fields."""
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam, w0 = 256, 2e-5, 1e-6, 4e-4
    zR = math.pi * w0 * w0 / lam                                 # 0.503 m
    x, y = coords(N, dx)
    u = np.exp(-(x * x + y * y) / w0 ** 2) * (1 + 0.1 * np.cos(2 * np.pi * x / 2e-4)) * np.exp(0.2j * np.sin(2 * np.pi * y / 3e-4))
    a, d, st, legs = oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, 0.2 * zR)], w0)
    assert np.array_equal(a, oracle.propagate_as(u, dx, lam, 0.2 * zR)) and legs == [(1, 0)]
    b, _, st2, _ = oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, 0.12 * zR), Surface(math.inf, 0.08 * zR)], w0)
    assert rel(b, a) <= 1e-13 and st2[2] == pytest.approx(0.2 * zR)
    z = 3.0 * zR
    s, d1, st, legs = oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, z)], w0)
    want, dxo = oracle.propagate_direct(u, dx, lam, z)
    assert legs == [(0, 2)] and d1 == dxo
    assert rel(true_field(s, d1, lam, st[3]), want) <= 1e-13
    # sphere -> sphere through the waist: from z = -3 zR to +2 zR
    st_in = (w0, 0.0, -z, -z)
    stored_in = u                                                # any stored array will do
    t, d2, st3, legs = oracle.system_run_pilot(stored_in, dx, lam, [Surface(math.inf, z + 2 * zR)], w0, state=st_in)
    assert legs == [(3, 2)] and st3[3] == pytest.approx(2 * zR)
    m, dm = oracle.propagate_direct(true_field(stored_in, dx, lam, -z), dx, lam, z)
    m, dm = oracle.propagate_direct(m, dm, lam, 2 * zR)
    assert d2 == pytest.approx(dm, rel=1e-14)
    assert rel(true_field(t, d2, lam, st3[3]), m) <= 1e-12
    # energy: sum |U|^2 dx^2 is conserved by every leg
    assert np.sum(np.abs(t) ** 2) * d2 ** 2 == pytest.approx(np.sum(np.abs(u) ** 2) * dx ** 2, rel=1e-12)


def test_P22_pilot_through_lenses_lands_on_the_abcd_closed_form(oracle):
    """Config 2 (Gaussian through three lenses) under the pilot-beam rule: after every surface the TRUE field equals
    the ABCD closed form of P5, the pilot state equals the closed-form beam (waist position and Rayleigh range from q),
    and the first propagation -- from a lens 0.499 m before its focus to 0.9 mm past it -- is STW then PTP."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config2()
    N, dx, lam, w0 = wl.N, float(wl.dx[0]), float(wl.lam[0]), 2e-3
    steps = [(s.f, s.z) for s in wl.surfaces]
    ref = abcd_chain(lam, w0, steps)
    u, d, st, zpos = wl.field[0], dx, None, 0.0
    for i, (s, (q, A)) in enumerate(zip(wl.surfaces, ref)):
        u, d, st, legs = oracle.system_run_pilot(u, d, lam, [s], w0, state=st)
        zpos += s.z
        if i == 0:
            assert legs == [(oracle.LEG_STW, oracle.LEG_PTP)]
        x, y = coords(N, d)
        assert rel(true_field(u, d, lam, st[3]), A * np.exp(1j * np.pi * (x * x + y * y) / (lam * q))) <= 1e-8, f"surface {i}"
        # closed-form beam: q = (z - zw) - i zR in the sign convention of abcd_chain
        assert st[2] == pytest.approx(zpos, rel=1e-14)
        assert st[2] - st[1] == pytest.approx(q.real, rel=1e-9, abs=1e-12)
        assert math.pi * st[0] ** 2 / lam == pytest.approx(-q.imag, rel=1e-9)
    assert st[0] == pytest.approx(math.sqrt(lam * 0.333305 / math.pi), rel=1e-5)       # zR = 0.333305 m after lens 3


def test_P23_pilot_masks_rayleigh_factor_and_errors(oracle):
    """Masks act on the stored array; the Rayleigh factor moves the planar/spherical boundary; a zero-length step and a
    z = 0 surface do nothing to the reference; bad arguments are refused."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam, w0 = 128, 2e-5, 1e-6, 3e-4
    zR = math.pi * w0 * w0 / lam
    u = rnd(N, 230)
    amp = inputs.circular_aperture(N, 40)
    opd = inputs.psd_map(N, dx, 3.0, 20e-9, 231)
    z = 1.5 * zR
    _, _, _, legs1 = oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, z)], w0, rayleigh_factor=1.0)
    _, _, _, legs2 = oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, z)], w0, rayleigh_factor=2.0)
    assert legs1 == [(0, 2)] and legs2 == [(1, 0)]
    a, d, st, legs = oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, 0.0, amp, opd), Surface(math.inf, z)], w0)
    b, d2 = oracle.wts(oracle.apply_mask(u, amp, opd, lam), dx, lam, z)
    assert legs == [(0, 0), (0, 2)] and d == d2 and np.array_equal(a, b)
    with pytest.raises(oracle.OracleError):
        oracle.system_run_pilot(u, dx, lam, [Surface(0.0, 0.1)], w0)
    with pytest.raises(oracle.OracleError):
        oracle.system_run_pilot(u, dx, lam, [Surface(math.inf, 0.1)], -1.0)


# ---- P24-P26: Fraunhofer matrix Fourier transform (reading g22) ----
def test_P24_mft_equals_the_centred_fft_at_critical_sampling(oracle):
    """At dx_out = lambda f/(na dx_in), nb = na the matrix transform IS the Fourier core of direct Fresnel:
    dx^2/(i lambda f) fftshift(fft2(ifftshift(U))) -- ties it to the pinned FFT (even, odd and non-power-of-two na);
    the inverse direction undoes it; and direct Fresnel itself is chirp x MFT x chirp."""
    lam, f = 0.8e-6, 0.7
    for na in (64, 45, 100):
        dx = 1.5e-5
        u = rnd(na, 240 + na)
        dxo = lam * f / (na * dx)
        v = oracle.mft(u, dx, na, dxo, lam, f, +1)
        want = dx * dx / (1j * lam * f) * np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(u)))
        assert rel(v, want) <= 1e-12
        assert rel(v, dx * dx / (1j * lam * f) * oracle.fft2d(u, +1, True)) <= 1e-12
        assert rel(oracle.mft(v, dxo, na, dx, lam, f, -1), u) <= 1e-12
    na, dx = 64, 1.5e-5
    u = rnd(na, 241)
    z = 0.4
    d, dxo = oracle.propagate_direct(u, dx, lam, z)
    m = oracle.mft(oracle.apply_qpf(u, dx, lam, z), dx, na, dxo, lam, z, +1)
    assert rel(oracle.apply_qpf(m, dxo, lam, z), d) <= 1e-12


def test_P24b_mft_on_a_coarser_grid_samples_the_centred_fft(oracle):
    """With an output pitch of s critical pixels the matrix transform lands on every s-th bin of the centred FFT around the
    centre bin: how tests/test_gpu_any_n.py takes single outputs of a 4100^2 transform from the oracle."""
    lam, f, dx = 0.8e-6, 0.7, 1.5e-5
    for na, nb, s in ((100, 9, 7), (45, 5, 4)):
        u = rnd(na, 245 + na)
        full = dx * dx / (1j * lam * f) * oracle.fft2d(u, +1, True)
        v = oracle.mft(u, dx, nb, s * lam * f / (na * dx), lam, f, +1)
        idx = na // 2 + (np.arange(nb) - nb // 2) * s
        assert rel(v, full[np.ix_(idx, idx)]) <= 1e-12


def test_P25_mft_closed_forms(oracle):
    """Closed forms on an output grid the FFT cannot reach (nb != na, 3.7x finer than critical): the centre sample is
    sum(U) dx^2/(i lambda f) exactly; a uniform square aperture gives the product of two Dirichlet kernels; a shifted
    delta gives a pure phase ramp of the right sign and slope; linearity and separability."""
    lam, f, na, dx, nb = 1e-6, 0.5, 48, 2e-5, 37
    dxo = lam * f / (na * dx) / 3.7
    u = rnd(na, 250)
    v = oracle.mft(u, dx, nb, dxo, lam, f, +1)
    assert v[nb // 2, nb // 2] == pytest.approx(u.sum() * dx * dx / (1j * lam * f), rel=1e-12)
    # square aperture of half-width h pixels (indices -h..h): sum_k exp(-2 pi i k a) = sin(pi (2h+1) a)/sin(pi a), a = dx x'/(lam f)
    h = 7
    sq = np.zeros((na, na))
    sq[na // 2 - h:na // 2 + h + 1, na // 2 - h:na // 2 + h + 1] = 1.0
    a = dx * (np.arange(nb) - nb // 2) * dxo / (lam * f)
    with np.errstate(invalid="ignore", divide="ignore"):
        dk = np.where(a == 0, 2 * h + 1, np.sin(np.pi * (2 * h + 1) * a) / np.sin(np.pi * a))
    want = dx * dx / (1j * lam * f) * dk[:, None] * dk[None, :]
    assert rel(oracle.mft(sq, dx, nb, dxo, lam, f, +1), want) <= 1e-12
    # delta at pixel (j0, k0): exp(-2 pi i (x_k0 x' + y_j0 y')/(lam f)) -- and the conjugate ramp for the inverse kernel
    j0, k0 = na // 2 + 5, na // 2 - 3
    d = np.zeros((na, na), complex)
    d[j0, k0] = 1.0
    xo = (np.arange(nb) - nb // 2) * dxo
    ramp = np.exp(-2j * np.pi * ((k0 - na // 2) * dx * xo[None, :] + (j0 - na // 2) * dx * xo[:, None]) / (lam * f))
    assert rel(oracle.mft(d, dx, nb, dxo, lam, f, +1), dx * dx / (1j * lam * f) * ramp) <= 1e-13
    assert rel(oracle.mft(d, dx, nb, dxo, lam, f, -1), dx * dx / (-1j * lam * f) * np.conj(ramp)) <= 1e-13
    w = rnd(na, 251)
    assert rel(oracle.mft(2.0 * u - 1j * w, dx, nb, dxo, lam, f, +1), 2.0 * v - 1j * oracle.mft(w, dx, nb, dxo, lam, f, +1)) <= 1e-13


def test_P26_mft_airy_pattern_oversampled(oracle):
    """The use the paper names (a coronagraph's focal plane at high sampling over a small field): circular aperture of
    radius a -> Airy amplitude (pi a^2/(lam f)) 2 J1(v)/v, v = 2 pi a r'/(lam f), sampled 8x finer than the FFT would,
    over +-3 Airy rings; the pixelated disc matches the continuous pattern to a fraction of a per cent of the peak
    (as P8), and the first null sits at 0.61 lam f / a."""
    from paper_1806_06467_b200 import inputs
    lam, f, na, dx = 1e-6, 0.5, 256, 1e-5
    a_px = 100
    ap = inputs.circular_aperture(na, a_px)
    nb = 96
    dxo = lam * f / (na * dx) / 8.0
    v = oracle.mft(ap, dx, nb, dxo, lam, f, +1)
    c = nb // 2
    assert v[c, c] == pytest.approx(ap.sum() * dx * dx / (1j * lam * f), rel=1e-12)
    xo = (np.arange(nb) - c) * dxo
    r = np.hypot(xo[None, :], xo[:, None])
    arg = 2 * np.pi * a_px * dx * r / (lam * f)
    with np.errstate(invalid="ignore", divide="ignore"):
        airy = np.where(arg == 0, 1.0, 2 * j1(arg) / arg)
    want = (np.pi * (a_px * dx) ** 2 / (lam * f)) * airy
    assert np.abs(np.abs(v) - np.abs(want)).max() <= 4e-3 * np.abs(want).max()
    prof = np.abs(v[c, c:])
    null_px = next(i for i in range(1, 40) if prof[i] < prof[i - 1] and prof[i] < prof[i + 1])      # first local minimum
    assert null_px == pytest.approx(0.6098 * lam * f / (a_px * dx) / dxo, abs=1.0)
