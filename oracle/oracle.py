"""ctypes face of oracle/liboracle.so (TEST INFRASTRUCTURE -- see fresnel_oracle.c header).

Every function takes/returns numpy complex128 arrays of shape (N, N) (or (batch, N, N) for the
``*_batch`` helpers, which just loop) and never touches the GPU.  Citations are in the C file.
"""
import ctypes
import math

import numpy as np

from . import build as _build

_lib = None

ORACLE_OK = 0
FORWARD = +1
INVERSE = -1


class OracleError(RuntimeError):
    pass


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        L.oracle_set_threads.argtypes = [ctypes.c_int]
        L.oracle_set_threads.restype = None
        L.oracle_get_threads.argtypes = []
        L.oracle_get_threads.restype = ctypes.c_int
        L.oracle_dft2_naive.argtypes = [dp, ctypes.c_int, ctypes.c_int]
        L.oracle_fft2.argtypes = [dp, ctypes.c_int, ctypes.c_int]
        L.oracle_dft2_any.argtypes = [dp, ctypes.c_int, ctypes.c_int]
        L.oracle_dft2_any.restype = ctypes.c_int
        L.oracle_fftshift.argtypes = [dp, ctypes.c_int]
        L.oracle_ifftshift.argtypes = [dp, ctypes.c_int]
        L.oracle_fft2d.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.oracle_apply_qpf.argtypes = [dp, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double]
        L.oracle_apply_mask.argtypes = [dp, ctypes.c_int, dp, dp, ctypes.c_double]
        L.oracle_propagate_as.argtypes = [dp, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double]
        L.oracle_propagate_direct.argtypes = [dp, ctypes.c_int, dp, ctypes.c_double, ctypes.c_double]
        L.oracle_surface_as.argtypes = [dp, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                        dp, dp, ctypes.c_double]
        pp = ctypes.POINTER(dp)
        L.oracle_system_run.argtypes = [dp, ctypes.c_int, dp, ctypes.c_double, ctypes.c_int, dp, pp, pp, dp,
                                        ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
        L.oracle_system_run.restype = ctypes.c_int
        L.oracle_wts.argtypes = [dp, ctypes.c_int, dp, ctypes.c_double, ctypes.c_double]
        L.oracle_wts.restype = ctypes.c_int
        L.oracle_stw.argtypes = [dp, ctypes.c_int, dp, ctypes.c_double, ctypes.c_double]
        L.oracle_stw.restype = ctypes.c_int
        L.oracle_system_run_pilot.argtypes = [dp, ctypes.c_int, dp, ctypes.c_double, ctypes.c_int, dp, pp, pp, dp,
                                              ctypes.c_double, dp, ctypes.POINTER(ctypes.c_int)]
        L.oracle_system_run_pilot.restype = ctypes.c_int
        L.oracle_mft.argtypes = [dp, ctypes.c_int, ctypes.c_double, dp, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int]
        L.oracle_mft.restype = ctypes.c_int
        L.oracle_accumulate_intensity.argtypes = [dp, ctypes.c_int, ctypes.c_double, dp]
        L.oracle_accumulate_intensity.restype = ctypes.c_int
        for name in ("oracle_dft2_naive", "oracle_fft2", "oracle_fftshift", "oracle_ifftshift", "oracle_fft2d",
                     "oracle_apply_qpf", "oracle_apply_mask", "oracle_propagate_as", "oracle_propagate_direct",
                     "oracle_surface_as"):
            getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def get_threads() -> int:
    return int(lib().oracle_get_threads())


def _prep(u):
    a = np.array(u, dtype=np.complex128, order="C", copy=True)
    if a.ndim != 2 or a.shape[0] != a.shape[1]:
        raise ValueError("oracle expects a square (N, N) array")
    return a, a.shape[0]


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _real(m, N):
    if m is None:
        return None, None
    a = np.ascontiguousarray(m, dtype=np.float64)
    if a.shape != (N, N):
        raise ValueError("map must be (N, N)")
    return a, _dptr(a)


def _check(rc, what):
    if rc != ORACLE_OK:
        raise OracleError(f"{what} failed with oracle status {rc}")


def dft2_naive(u, sign):
    a, N = _prep(u)
    _check(lib().oracle_dft2_naive(_dptr(a), N, int(sign)), "dft2_naive")
    return a


def fft2(u, sign):
    a, N = _prep(u)
    _check(lib().oracle_fft2(_dptr(a), N, int(sign)), "fft2")
    return a


def dft2_any(u, sign):
    """The plain separable O(N^3) DFT, any N (what fft2 uses when N is not a power of two)."""
    a, N = _prep(u)
    _check(lib().oracle_dft2_any(_dptr(a), N, int(sign)), "dft2_any")
    return a


def fftshift(u):
    a, N = _prep(u)
    _check(lib().oracle_fftshift(_dptr(a), N), "fftshift")
    return a


def ifftshift(u):
    a, N = _prep(u)
    _check(lib().oracle_ifftshift(_dptr(a), N), "ifftshift")
    return a


def fft2d(u, direction, centered):
    a, N = _prep(u)
    _check(lib().oracle_fft2d(_dptr(a), N, int(direction), int(bool(centered))), "fft2d")
    return a


def apply_qpf(u, dx, lam, z):
    a, N = _prep(u)
    _check(lib().oracle_apply_qpf(_dptr(a), N, float(dx), float(lam), float(z)), "apply_qpf")
    return a


def apply_mask(u, amp, opd, lam):
    a, N = _prep(u)
    ka, pa = _real(amp, N)
    ko, po = _real(opd, N)
    _check(lib().oracle_apply_mask(_dptr(a), N, pa, po, float(lam)), "apply_mask")
    return a


def propagate_as(u, dx, lam, z):
    a, N = _prep(u)
    _check(lib().oracle_propagate_as(_dptr(a), N, float(dx), float(lam), float(z)), "propagate_as")
    return a


def propagate_direct(u, dx, lam, z):
    """Returns (field, dx_out)."""
    a, N = _prep(u)
    d = ctypes.c_double(float(dx))
    _check(lib().oracle_propagate_direct(_dptr(a), N, ctypes.byref(d), float(lam), float(z)), "propagate_direct")
    return a, d.value


def surface_as(u, dx, lam, f, amp, opd, z):
    a, N = _prep(u)
    ka, pa = _real(amp, N)
    ko, po = _real(opd, N)
    _check(lib().oracle_surface_as(_dptr(a), N, float(dx), float(lam),
                                   float(f) if f is not None else math.inf, pa, po, float(z)), "surface_as")
    return a


# -- batch helpers: the batch dimension is just a loop over independent wavefronts --

def _per_batch(x, b):
    arr = np.atleast_1d(np.asarray(x, dtype=np.float64))
    return float(arr[b] if arr.size > 1 else arr[0])


def propagate_as_batch(u, dx, lam, z):
    u = np.asarray(u)
    return np.stack([propagate_as(u[b], _per_batch(dx, b), _per_batch(lam, b), z) for b in range(u.shape[0])])


def surface_as_batch(u, dx, lam, f, amp, opd, z):
    u = np.asarray(u)
    return np.stack([surface_as(u[b], _per_batch(dx, b), _per_batch(lam, b), f, amp, opd, z)
                     for b in range(u.shape[0])])


def accumulate_intensity(u, w, image=None):
    """image += w * |u|^2 (NEXT-3).  u: (N, N) complex; returns the (N, N) float64 image."""
    a = np.ascontiguousarray(np.asarray(u, dtype=np.complex128))
    N = a.shape[-1]
    img = np.zeros((N, N)) if image is None else np.ascontiguousarray(np.asarray(image, dtype=np.float64)).copy()
    _check(lib().oracle_accumulate_intensity(_dptr(a), N, float(w), img.ctypes.data_as(ctypes.POINTER(ctypes.c_double))),
           "accumulate_intensity")
    return img


def broadband_image(u, weights):
    """sum_b weights[b] * |u[b]|^2 for a (batch, N, N) stack of monochromatic fields."""
    u = np.asarray(u)
    img = np.zeros(u.shape[-2:])
    for b in range(u.shape[0]):
        img = accumulate_intensity(u[b], float(np.asarray(weights)[b]), img)
    return img


METHOD_AS, METHOD_DIRECT, METHOD_AUTO = 0, 1, 2


def system_run(u, dx, lam, surfaces, methods=None):
    """Train of surfaces on one wavefront (NEXT-1 reduced, reading g13b).  `surfaces`: objects
    with .f (None/inf = no lens), .amp, .opd, .z; `methods`: per-surface 0/1/2 (default AUTO).
    Returns (field, final pixel pitch, list of methods used: 0 AS, 1 direct, -1 none)."""
    a, N = _prep(u)
    n = len(surfaces)
    dp = ctypes.POINTER(ctypes.c_double)
    f = np.array([math.inf if s.f is None else float(s.f) for s in surfaces], dtype=np.float64)
    z = np.array([float(s.z) for s in surfaces], dtype=np.float64)
    m = np.array([METHOD_AUTO] * n if methods is None else list(methods), dtype=np.int32)
    keep, amp_p, opd_p = [], (dp * max(n, 1))(), (dp * max(n, 1))()
    for i, s in enumerate(surfaces):
        ka, pa = _real(s.amp, N)
        ko, po = _real(s.opd, N)
        keep += [ka, ko]
        amp_p[i] = pa if pa is not None else ctypes.cast(None, dp)
        opd_p[i] = po if po is not None else ctypes.cast(None, dp)
    dxv = ctypes.c_double(float(dx))
    used = np.zeros(max(n, 1), dtype=np.int32)
    _check(lib().oracle_system_run(_dptr(a), N, ctypes.byref(dxv), float(lam), n, f.ctypes.data_as(dp), amp_p, opd_p,
                                   z.ctypes.data_as(dp), m.ctypes.data_as(ctypes.POINTER(ctypes.c_int)),
                                   used.ctypes.data_as(ctypes.POINTER(ctypes.c_int))), "system_run")
    return a, dxv.value, [int(x) for x in used[:n]]


def wts(u, dx, lam, dz):
    """Waist -> spherical (direct Fresnel without its output chirp).  Returns (stored field, dx_out)."""
    a, N = _prep(u)
    d = ctypes.c_double(float(dx))
    _check(lib().oracle_wts(_dptr(a), N, ctypes.byref(d), float(lam), float(dz)), "wts")
    return a, d.value


def stw(u, dx, lam, dz):
    """Spherical -> waist (direct Fresnel without its input chirp).  Returns (field, dx_out)."""
    a, N = _prep(u)
    d = ctypes.c_double(float(dx))
    _check(lib().oracle_stw(_dptr(a), N, ctypes.byref(d), float(lam), float(dz)), "stw")
    return a, d.value


LEG_NONE, LEG_PTP, LEG_WTS, LEG_STW = 0, 1, 2, 3


def system_run_pilot(u, dx, lam, surfaces, w0, rayleigh_factor=1.0, state=None):
    """Train of surfaces under the Gaussian pilot-beam rule (NEXT-1; conventions in fresnel_oracle.c).  `state`:
    (w0, zw, z, Rref) to continue from, default a waist of radius w0 at z = 0 on a planar reference.
    Returns (stored field, final pixel pitch, state tuple (w0, zw, z, Rref), legs [(leg1, leg2), ...])."""
    a, N = _prep(u)
    n = len(surfaces)
    dp = ctypes.POINTER(ctypes.c_double)
    f = np.array([math.inf if s.f is None else float(s.f) for s in surfaces], dtype=np.float64)
    z = np.array([float(s.z) for s in surfaces], dtype=np.float64)
    keep, amp_p, opd_p = [], (dp * max(n, 1))(), (dp * max(n, 1))()
    for i, s in enumerate(surfaces):
        ka, pa = _real(s.amp, N)
        ko, po = _real(s.opd, N)
        keep += [ka, ko]
        amp_p[i] = pa if pa is not None else ctypes.cast(None, dp)
        opd_p[i] = po if po is not None else ctypes.cast(None, dp)
    dxv = ctypes.c_double(float(dx))
    st = np.array([float(w0), 0.0, 0.0, math.inf, 0.0] if state is None else list(state) + [0.0], dtype=np.float64)
    legs = np.zeros(2 * max(n, 1), dtype=np.int32)
    _check(lib().oracle_system_run_pilot(_dptr(a), N, ctypes.byref(dxv), float(lam), n, f.ctypes.data_as(dp), amp_p, opd_p,
                                         z.ctypes.data_as(dp), float(rayleigh_factor), st.ctypes.data_as(dp),
                                         legs.ctypes.data_as(ctypes.POINTER(ctypes.c_int))), "system_run_pilot")
    return a, dxv.value, tuple(float(x) for x in st[:4]), [(int(legs[2 * i]), int(legs[2 * i + 1])) for i in range(n)]


def mft(u, dx_in, nb, dx_out, lam, f, direction=+1):
    """Fraunhofer propagation by a matrix Fourier transform onto an nb x nb grid of pitch dx_out (NEXT-4)."""
    a, na = _prep(u)
    out = np.zeros((int(nb), int(nb)), dtype=np.complex128)
    _check(lib().oracle_mft(_dptr(a), na, float(dx_in), _dptr(out), int(nb), float(dx_out), float(lam), float(f), int(direction)), "mft")
    return out
