"""Seeded synthetic input generators -- the ONLY module shared by the oracle tests and the CUDA path.

It holds none of the method's arithmetic: no chirp, no transfer function, no propagation.  It only
draws random numbers (numpy ``Generator(PCG64(seed))``) and shapes them into the workloads that
BASELINE.json:configs name (recipes restated in DESIGN.md, "Input recipe").  These inputs STAND IN
for the paper's WFIRST shaped-pupil-coronagraph model, whose FITS inputs
(WebbPSF data 0.7.0) are not available and are not recreated.

numpy's FFT is used here for one thing only: colouring white noise into a power-law PSD surface
map (an input, not a step of the method).  It is in neither timed path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def centred_r2_px(N: int) -> np.ndarray:
    """(j-N/2)^2 + (k-N/2)^2 in pixels^2 (origin on pixel N/2, reading g8)."""
    c = np.arange(N, dtype=np.float64) - N // 2
    return c[:, None] ** 2 + c[None, :] ** 2


def circular_aperture(N: int, radius_px: float) -> np.ndarray:
    """1 where (j-N/2)^2+(k-N/2)^2 <= R^2 (inclusive, reading g9), else 0."""
    return (centred_r2_px(N) <= radius_px * radius_px).astype(np.float64)


def psd_map(N: int, dx: float, power: float, rms: float, seed: int, support: Optional[np.ndarray] = None) -> np.ndarray:
    """Random surface map with a |f|^-power power spectral density (own formulation):
    white noise -> FFT2 -> x |f|^(-power/2), DC removed -> real part of IFFT2 -> zero mean and the
    stated RMS over ``support`` (default: the whole grid); zero outside ``support``."""
    g = _rng(seed).standard_normal((N, N))
    G = np.fft.fft2(g)
    f = np.fft.fftfreq(N, d=dx)
    fr = np.sqrt(f[:, None] ** 2 + f[None, :] ** 2)
    fr[0, 0] = 1.0
    G *= fr ** (-power / 2.0)
    G[0, 0] = 0.0
    m = np.fft.ifft2(G).real
    if support is None:
        m -= m.mean()
        m *= rms / math.sqrt(np.mean(m * m))
    else:
        sel = support > 0
        m -= m[sel].mean()
        m *= rms / math.sqrt(np.mean(m[sel] ** 2))
        m = np.where(sel, m, 0.0)
    return np.ascontiguousarray(m)


def random_field(N: int, seed: int, batch: int = 1) -> np.ndarray:
    """real, imag ~ N(0,1) i.i.d. (config 4)."""
    r = _rng(seed)
    u = r.standard_normal((batch, N, N)) + 1j * r.standard_normal((batch, N, N))
    return np.ascontiguousarray(u.astype(np.complex128))


# --------------------------------------------------------------------------------------------
# BASELINE.json:configs restated as concrete synthetic inputs
# --------------------------------------------------------------------------------------------

@dataclass
class Surface:
    """One optical surface followed by a propagation: thin lens f (inf = none), optional amplitude
    and OPD maps (metres), then distance z."""
    f: float
    z: float
    amp: Optional[np.ndarray] = None
    opd: Optional[np.ndarray] = None


@dataclass
class Workload:
    name: str
    N: int
    dtype: str                 # "c128" | "c64"
    field: np.ndarray          # (batch, N, N) complex128 (cast to complex64 by the caller for c64)
    dx: np.ndarray             # (batch,) metres
    lam: np.ndarray            # (batch,) metres
    surfaces: List[Surface] = field(default_factory=list)

    @property
    def batch(self) -> int:
        return self.field.shape[0]


def config1() -> Workload:
    """256x256 c128, unit-amplitude circular aperture R=64 px, phase ~ N(0, 0.05 rad), one AS step."""
    N = 256
    ap = circular_aperture(N, 64)
    phi = _rng(1001).normal(0.0, 0.05, size=(N, N))
    u = ap * np.exp(1j * phi)
    return Workload("cfg1_as_256_c128", N, "c128", u[None].astype(np.complex128),
                    np.array([1e-4]), np.array([1e-6]), [Surface(math.inf, 0.1)])


def config2() -> Workload:
    """1024x1024 c128 Gaussian beam, waist 2 mm, 3 thin lenses f=.5,.25,1 separated by z=.5,.75,1."""
    N, dx, w0 = 1024, 2e-5, 2e-3
    r2 = centred_r2_px(N) * dx * dx
    u = np.exp(-r2 / (w0 * w0))
    surfs = [Surface(0.5, 0.5), Surface(0.25, 0.75), Surface(1.0, 1.0)]
    return Workload("cfg2_gauss_1024_c128", N, "c128", u[None].astype(np.complex128),
                    np.array([dx]), np.array([1.064e-6]), surfs)


def config3(N: int = 2048, n_surfaces: int = 20) -> Workload:
    """Shaped-pupil-coronagraph analog: N=2048 c128, lambda=550 nm, dx=2e-5 (pupil radius N/8 px),
    20 surfaces each = thin lens f~U[0.2,3] + f^-3 PSD OPD map at 10 nm RMS + z~U[0.1,2];
    circular pupil on surface 0, binary shaped pupil on 6, occulting disk on 12 (reading g17).
    ``N`` may be reduced for parity tests (pupil and masks scale with N/2048)."""
    dx, lam = 2e-5, 550e-9
    s = N / 2048.0
    r = _rng(3000)
    fs = r.uniform(0.2, 3.0, size=20)
    zs = r.uniform(0.1, 2.0, size=20)
    pupil = circular_aperture(N, 256 * s)
    surfs = []
    for i in range(n_surfaces):
        opd = psd_map(N, dx, 3.0, 10e-9, 3100 + i)
        amp = None
        if i == 0:
            amp = pupil
        elif i == 6:
            blk = max(1, int(round(8 * s)))
            bits = (_rng(3200).random((64, 64)) < 0.5).astype(np.float64)
            tile = np.kron(bits, np.ones((blk, blk)))
            amp = np.zeros((N, N))
            h = tile.shape[0] // 2
            amp[N // 2 - h:N // 2 + h, N // 2 - h:N // 2 + h] = tile
            amp *= pupil
        elif i == 12:
            amp = (centred_r2_px(N) > (24 * s) ** 2).astype(np.float64)
        surfs.append(Surface(float(fs[i]), float(zs[i]), amp, opd))
    u = np.ones((1, N, N), dtype=np.complex128)
    return Workload(f"cfg3_spc_{N}_c128", N, "c128", u, np.array([dx]), np.array([lam]), surfs)


def config4(N: int, dtype: str) -> Workload:
    """Single AS step of a complex Gaussian-random field, lambda=1e-6, z=0.5, dx=1e-5."""
    seed = 4000 + int(round(math.log2(N)))
    u = random_field(N, seed)
    if dtype == "c64":
        u = u.astype(np.complex64).astype(np.complex128)   # the float32 cast IS the input for both paths
    return Workload(f"cfg4_as_{N}_{dtype}", N, dtype, u, np.array([1e-5]), np.array([1e-6]),
                    [Surface(math.inf, 0.5)])


def config5(N: int = 4096, batch: int = 16, planes: int = 10) -> Workload:
    """Polychromatic batch: ``batch`` wavelengths evenly spaced 500-600 nm, N=4096 c64, circular
    pupil radius N/8 px with an f^-2.5 PSD OPD at 20 nm RMS over the pupil, 10 planes of
    (thin lens f=1 m + z=0.3 m).  dx=1e-5 (reading g18)."""
    dx = 1e-5
    lam = 500e-9 + np.arange(batch) * (100e-9 / max(batch - 1, 1))
    pupil = circular_aperture(N, N / 8)
    opd = psd_map(N, dx, 2.5, 20e-9, 5001, support=pupil)
    surfs = [Surface(1.0, 0.3, pupil, opd)] + [Surface(1.0, 0.3) for _ in range(planes - 1)]
    u = np.ones((batch, N, N), dtype=np.complex128)
    return Workload(f"cfg5_poly_{N}_c64_b{batch}", N, "c64", u, np.full(batch, dx), lam, surfs)
