"""Thin ctypes face of libfresnel.so (the C ABI declared in include/fresnel.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  torch is
used for device memory and streams, nothing else.  There is NO fallback: if libfresnel.so is
missing or a call fails, an exception is raised.

    plan = Plan(N=2048, batch=1, dtype="c128")
    plan.surface_as(wf, pixel=[2e-5], lam=[550e-9], f=0.5, amp=amp, opd=opd, z=0.3)   # in place
"""
from __future__ import annotations

import ctypes
import math
import os
from typing import Optional, Sequence

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FRESNEL_LIB", os.path.join(HERE, "libfresnel.so"))   # override: tuning builds only

FRESNEL_OK = 0
FORWARD = +1
INVERSE = -1
C64, C128 = 0, 1

# every symbol include/fresnel.h declares (tests/test_abi.py checks the header against this list)
SYMBOLS = (
    "fresnel_plan_create", "fresnel_plan_set_stream", "fresnel_plan_synchronize", "fresnel_plan_destroy",
    "fresnel_plan_launch_count", "fresnel_plan_record_pass_events", "fresnel_plan_record_train_events",
    "fresnel_plan_last_schedule", "fresnel_plan_reserve_tables", "fresnel_plan_release_graph_tables", "fresnel_apply_qpf", "fresnel_apply_mask", "fresnel_fft2d",
    "fresnel_propagate_as", "fresnel_propagate_direct", "fresnel_surface_as", "fresnel_system_run", "fresnel_system_run_pilot", "fresnel_plan_reserve_mft", "fresnel_mft", "fresnel_mft_noalloc", "fresnel_accumulate_intensity", "fresnel_memcpy_h2d",
    "fresnel_memcpy_d2h", "fresnel_status_string", "fresnel_version",
)

_lib = None

METHOD_AS, METHOD_DIRECT, METHOD_AUTO = 0, 1, 2


class _Surface(ctypes.Structure):       # fresnel_surface of include/fresnel.h
    _fields_ = [("f", ctypes.c_double), ("amp", ctypes.c_void_p), ("opd", ctypes.c_void_p),
                ("z", ctypes.c_double), ("method", ctypes.c_int)]


class _PilotState(ctypes.Structure):   # fresnel_pilot_state of include/fresnel.h
    _fields_ = [("w0", ctypes.c_double), ("zw", ctypes.c_double), ("z", ctypes.c_double), ("rref", ctypes.c_double)]


LEG_NONE, LEG_PTP, LEG_WTS, LEG_STW = 0, 1, 2, 3


class _PassInfo(ctypes.Structure):      # fresnel_pass_info of include/fresnel.h
    _fields_ = [("direction", ctypes.c_int), ("convolutions", ctypes.c_int), ("first_surface", ctypes.c_int),
                ("maps_read", ctypes.c_int)]


class FresnelError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        name = lib().fresnel_status_string(status).decode() if _lib is not None else str(status)
        super().__init__(f"{what}: {name}")


def lib() -> ctypes.CDLL:
    """Load libfresnel.so; fails loudly when the CUDA extension has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1806_06467_b200.build` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, ci, cd = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double
    L.fresnel_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci]
    L.fresnel_plan_set_stream.argtypes = [vp, vp]
    L.fresnel_plan_synchronize.argtypes = [vp]
    L.fresnel_plan_destroy.argtypes = [vp]
    L.fresnel_plan_launch_count.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
    L.fresnel_plan_record_pass_events.argtypes = [vp, ctypes.POINTER(vp)]
    L.fresnel_plan_record_train_events.argtypes = [vp, ctypes.POINTER(vp), ci]
    L.fresnel_plan_last_schedule.argtypes = [vp, ctypes.POINTER(_PassInfo), ci, ctypes.POINTER(ci)]
    L.fresnel_plan_reserve_tables.argtypes = [vp, ci]
    L.fresnel_plan_release_graph_tables.argtypes = [vp]
    L.fresnel_apply_qpf.argtypes = [vp, vp, dp, dp, cd]
    L.fresnel_apply_mask.argtypes = [vp, vp, vp, vp, dp]
    L.fresnel_fft2d.argtypes = [vp, vp, ci, ci]
    L.fresnel_propagate_as.argtypes = [vp, vp, dp, dp, cd]
    L.fresnel_propagate_direct.argtypes = [vp, vp, dp, dp, cd]
    L.fresnel_surface_as.argtypes = [vp, vp, dp, dp, cd, vp, vp, cd]
    L.fresnel_system_run.argtypes = [vp, vp, dp, dp, ctypes.POINTER(_Surface), ci, ctypes.POINTER(ci)]
    L.fresnel_system_run_pilot.argtypes = [vp, vp, dp, dp, ctypes.POINTER(_Surface), ci, cd, ctypes.POINTER(_PilotState), ctypes.POINTER(ci)]
    L.fresnel_plan_reserve_mft.argtypes = [vp, ci]
    L.fresnel_mft.argtypes = [vp, vp, vp, ci, dp, dp, dp, cd, ci]
    L.fresnel_mft_noalloc.argtypes = [vp, vp, ci, ci, ci, ci, dp, dp, dp, cd, ci, vp]
    L.fresnel_accumulate_intensity.argtypes = [vp, vp, dp, vp]
    L.fresnel_memcpy_h2d.argtypes = [vp, vp, vp, ctypes.c_size_t]
    L.fresnel_memcpy_d2h.argtypes = [vp, vp, vp, ctypes.c_size_t]
    for s in SYMBOLS:
        getattr(L, s).restype = ci
    L.fresnel_status_string.argtypes = [ci]
    L.fresnel_status_string.restype = ctypes.c_char_p
    L.fresnel_version.argtypes = []
    L.fresnel_version.restype = ctypes.c_char_p
    _lib = L
    return L


def version() -> str:
    return lib().fresnel_version().decode()


def _darr(x, n: int):
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(x, dtype=np.float64), (n,)))
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


class Plan:
    """A fresnel_plan: N x N grids, `batch` wavefronts, dtype "c64" or "c128"."""

    def __init__(self, N: int, batch: int = 1, dtype: str = "c128", stream=None):
        import torch
        self._torch = torch
        self.N, self.batch, self.dtype = int(N), int(batch), dtype
        code = {"c64": C64, "c128": C128}.get(dtype)
        if code is None:
            raise ValueError("dtype must be 'c64' or 'c128'")
        self.cdtype = torch.complex64 if dtype == "c64" else torch.complex128
        self.rdtype = torch.float32 if dtype == "c64" else torch.float64
        self._h = ctypes.c_void_p()
        st = lib().fresnel_plan_create(ctypes.byref(self._h), self.N, self.batch, code)
        if st != FRESNEL_OK:
            self._h = ctypes.c_void_p()
            raise FresnelError(st, "fresnel_plan_create")
        if stream is None:
            stream = torch.cuda.current_stream()
        self.set_stream(stream)

    # -- plumbing ------------------------------------------------------------------------------
    def set_stream(self, stream) -> None:
        self._stream = stream
        self._chk(lib().fresnel_plan_set_stream(self._h, ctypes.c_void_p(stream.cuda_stream)), "fresnel_plan_set_stream")

    def synchronize(self) -> None:
        self._chk(lib().fresnel_plan_synchronize(self._h), "fresnel_plan_synchronize")

    def launch_count(self) -> int:
        c = ctypes.c_ulonglong(0)
        self._chk(lib().fresnel_plan_launch_count(self._h, ctypes.byref(c)), "fresnel_plan_launch_count")
        return int(c.value)

    def record_pass_events(self, events) -> None:
        """Arm the profiling hook with 3 torch.cuda.Event(enable_timing=True) objects (or None)."""
        if events is None:
            self._chk(lib().fresnel_plan_record_pass_events(self._h, None), "fresnel_plan_record_pass_events")
            return
        for e in events:
            if not e.cuda_event:          # torch creates the handle lazily on first record()
                e.record(self._stream)
        arr = (ctypes.c_void_p * 3)(*[ctypes.c_void_p(e.cuda_event) for e in events])
        self._chk(lib().fresnel_plan_record_pass_events(self._h, arr), "fresnel_plan_record_pass_events")

    def record_train_events(self, events) -> None:
        """Arm the train profiling hook: the next system_run records events[k] before its k-th pass kernel and one
        more after the last (torch.cuda.Event(enable_timing=True) objects; None or [] disarms)."""
        if not events:
            self._chk(lib().fresnel_plan_record_train_events(self._h, None, 0), "fresnel_plan_record_train_events")
            return
        for e in events:
            if not e.cuda_event:
                e.record(self._stream)
        arr = (ctypes.c_void_p * len(events))(*[ctypes.c_void_p(e.cuda_event) for e in events])
        self._chk(lib().fresnel_plan_record_train_events(self._h, arr, len(events)), "fresnel_plan_record_train_events")

    def last_schedule(self):
        """Pass kernels of the last system_run: list of dicts (direction, convolutions, first_surface, maps_read)."""
        n = ctypes.c_int(0)
        self._chk(lib().fresnel_plan_last_schedule(self._h, None, 0, ctypes.byref(n)), "fresnel_plan_last_schedule")
        arr = (_PassInfo * max(n.value, 1))()
        self._chk(lib().fresnel_plan_last_schedule(self._h, arr, n.value, ctypes.byref(n)), "fresnel_plan_last_schedule")
        return [{"direction": arr[i].direction, "convolutions": arr[i].convolutions,
                 "first_surface": arr[i].first_surface, "maps_read": arr[i].maps_read} for i in range(n.value)]

    def reserve_tables(self, n: int) -> None:
        self._chk(lib().fresnel_plan_reserve_tables(self._h, int(n)), "fresnel_plan_reserve_tables")

    def release_graph_tables(self) -> None:
        self._chk(lib().fresnel_plan_release_graph_tables(self._h), "fresnel_plan_release_graph_tables")

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().fresnel_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, st: int, what: str) -> None:
        if st != FRESNEL_OK:
            raise FresnelError(st, what)

    def _wf(self, wf) -> ctypes.c_void_p:
        if wf.dtype != self.cdtype or not wf.is_cuda or not wf.is_contiguous():
            raise ValueError(f"wavefront must be a contiguous CUDA tensor of {self.cdtype}")
        if wf.numel() != self.batch * self.N * self.N:
            raise ValueError("wavefront must have batch*N*N elements")
        return ctypes.c_void_p(wf.data_ptr())

    def _map(self, m) -> ctypes.c_void_p:
        if m is None:
            return ctypes.c_void_p(None)
        if m.dtype != self.rdtype or not m.is_cuda or not m.is_contiguous() or m.numel() != self.N * self.N:
            raise ValueError(f"maps must be contiguous CUDA tensors of {self.rdtype} with N*N elements")
        return ctypes.c_void_p(m.data_ptr())

    # -- the C ABI, same names -------------------------------------------------------------------
    def apply_qpf(self, wf, pixel, lam, z: float) -> None:
        _, pp = _darr(pixel, self.batch)
        _, lp = _darr(lam, self.batch)
        self._chk(lib().fresnel_apply_qpf(self._h, self._wf(wf), pp, lp, float(z)), "fresnel_apply_qpf")

    def apply_mask(self, wf, amp, opd, lam) -> None:
        _, lp = _darr(lam, self.batch)
        self._chk(lib().fresnel_apply_mask(self._h, self._wf(wf), self._map(amp), self._map(opd), lp), "fresnel_apply_mask")

    def fft2d(self, wf, direction: int = FORWARD, centered: bool = False) -> None:
        self._chk(lib().fresnel_fft2d(self._h, self._wf(wf), int(direction), int(bool(centered))), "fresnel_fft2d")

    def propagate_as(self, wf, pixel, lam, z: float) -> None:
        _, pp = _darr(pixel, self.batch)
        _, lp = _darr(lam, self.batch)
        self._chk(lib().fresnel_propagate_as(self._h, self._wf(wf), pp, lp, float(z)), "fresnel_propagate_as")

    def propagate_direct(self, wf, pixel, lam, z: float) -> np.ndarray:
        """Returns the new pixel pitch per batch element."""
        pa, pp = _darr(pixel, self.batch)
        pa = pa.copy()
        pp = pa.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        _, lp = _darr(lam, self.batch)
        self._chk(lib().fresnel_propagate_direct(self._h, self._wf(wf), pp, lp, float(z)), "fresnel_propagate_direct")
        return pa

    def surface_as(self, wf, pixel, lam, f: Optional[float], amp, opd, z: float) -> None:
        _, pp = _darr(pixel, self.batch)
        _, lp = _darr(lam, self.batch)
        ff = math.inf if f is None else float(f)
        self._chk(lib().fresnel_surface_as(self._h, self._wf(wf), pp, lp, ff, self._map(amp), self._map(opd), float(z)),
                  "fresnel_surface_as")

    def system_run(self, wf, pixel, lam, surfaces, maps=None, methods=None):
        """Train of surfaces in one call.  surfaces: objects with .f, .z; maps[i] = (amp, opd) device tensors or
        None; methods: per-surface METHOD_AS / METHOD_DIRECT / METHOD_AUTO (default AUTO).
        Returns (final pixel pitch per batch element, methods used)."""
        n = len(surfaces)
        arr = (_Surface * max(n, 1))()
        for i, s in enumerate(surfaces):
            amp, opd = (maps[i] if maps is not None else (None, None))
            arr[i].f = math.inf if s.f is None else float(s.f)
            arr[i].amp = self._map(amp).value
            arr[i].opd = self._map(opd).value
            arr[i].z = float(s.z)
            arr[i].method = METHOD_AUTO if methods is None else int(methods[i])
        pa, _ = _darr(pixel, self.batch)
        pa = pa.copy()
        pp = pa.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        _, lp = _darr(lam, self.batch)
        used = (ctypes.c_int * max(n, 1))()
        self._chk(lib().fresnel_system_run(self._h, self._wf(wf), pp, lp, arr, n, used), "fresnel_system_run")
        return pa, [int(used[i]) for i in range(n)]

    def system_run_pilot(self, wf, pixel, lam, surfaces, w0, maps=None, rayleigh_factor: float = 1.0, state=None):
        """Train of surfaces under the Gaussian pilot-beam rule.  w0: pilot waist radius at the start (scalar or per
        batch element); state: list of (w0, zw, z, rref) per batch element to continue from (default: at the waist, z = 0,
        planar).  Returns (final pixel pitch per batch element, list of states, legs [(leg1, leg2), ...] per surface)."""
        n = len(surfaces)
        arr = (_Surface * max(n, 1))()
        for i, s in enumerate(surfaces):
            amp, opd = (maps[i] if maps is not None else (None, None))
            arr[i].f = math.inf if s.f is None else float(s.f)
            arr[i].amp = self._map(amp).value
            arr[i].opd = self._map(opd).value
            arr[i].z = float(s.z)
            arr[i].method = METHOD_AUTO
        pa, _ = _darr(pixel, self.batch)
        pa = pa.copy()
        pp = pa.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        _, lp = _darr(lam, self.batch)
        st = (_PilotState * self.batch)()
        w0a, _ = _darr(w0, self.batch)
        for b in range(self.batch):
            if state is None:
                st[b].w0, st[b].zw, st[b].z, st[b].rref = float(w0a[b]), 0.0, 0.0, math.inf
            else:
                st[b].w0, st[b].zw, st[b].z, st[b].rref = (float(x) for x in state[b])
        legs = (ctypes.c_int * (2 * max(n, 1)))()
        self._chk(lib().fresnel_system_run_pilot(self._h, self._wf(wf), pp, lp, arr, n, float(rayleigh_factor), st, legs),
                  "fresnel_system_run_pilot")
        return pa, [(st[b].w0, st[b].zw, st[b].z, st[b].rref) for b in range(self.batch)], [(int(legs[2 * i]), int(legs[2 * i + 1])) for i in range(n)]

    def reserve_mft(self, nb_max: int) -> None:
        self._chk(lib().fresnel_plan_reserve_mft(self._h, int(nb_max)), "fresnel_plan_reserve_mft")

    def mft(self, wf, out, pixel_in, pixel_out, lam, f: float, direction: int = FORWARD) -> None:
        """Fraunhofer matrix Fourier transform of wf ([batch][N][N]) onto out ([batch][nb][nb], same dtype)."""
        nb = int(out.shape[-1])
        if out.dtype != self.cdtype or not out.is_cuda or not out.is_contiguous() or out.numel() != self.batch * nb * nb:
            raise ValueError("out must be a contiguous CUDA tensor [batch][nb][nb] of the plan's dtype")
        _, pi = _darr(pixel_in, self.batch)
        _, po = _darr(pixel_out, self.batch)
        _, lp = _darr(lam, self.batch)
        self._chk(lib().fresnel_mft(self._h, self._wf(wf), ctypes.c_void_p(out.data_ptr()), nb, pi, po, lp, float(f), int(direction)),
                  "fresnel_mft")

    def accumulate_intensity(self, wf, weight, image) -> None:
        """image += sum_b weight[b] * |wf[b]|^2 (image: real N x N device tensor of the plan's precision)."""
        _, wp = _darr(weight, self.batch)
        self._chk(lib().fresnel_accumulate_intensity(self._h, self._wf(wf), wp, self._map(image)), "fresnel_accumulate_intensity")

    def memcpy_h2d(self, dst, src_host) -> None:
        nbytes = src_host.numel() * src_host.element_size()
        self._chk(lib().fresnel_memcpy_h2d(self._h, ctypes.c_void_p(dst.data_ptr()), ctypes.c_void_p(src_host.data_ptr()), nbytes),
                  "fresnel_memcpy_h2d")

    def memcpy_d2h(self, dst_host, src) -> None:
        nbytes = src.numel() * src.element_size()
        self._chk(lib().fresnel_memcpy_d2h(self._h, ctypes.c_void_p(dst_host.data_ptr()), ctypes.c_void_p(src.data_ptr()), nbytes),
                  "fresnel_memcpy_d2h")


MFT_NOALLOC_MAX_ELEMS, MFT_NOALLOC_MAX_BATCH = 262144, 32      # FRESNEL_MFT_NOALLOC_MAX_* of include/fresnel.h


def mft_noalloc(wf, out, pixel_in, pixel_out, lam, f: float, direction: int = FORWARD, stream=None) -> None:
    """fresnel_mft_noalloc: the matrix Fourier transform without a plan and without any device allocation (its scratch is
    a fixed array inside the library: batch * nb * na <= MFT_NOALLOC_MAX_ELEMS, batch <= MFT_NOALLOC_MAX_BATCH; calls that
    overlap on the GPU race on it).  wf: CUDA tensor [batch][na][na] complex64 / complex128, out: [batch][nb][nb], same dtype."""
    import torch
    if wf.dtype not in (torch.complex64, torch.complex128) or out.dtype != wf.dtype:
        raise ValueError("wf and out must be complex64 or complex128 tensors of the same dtype")
    if not (wf.is_cuda and out.is_cuda and wf.is_contiguous() and out.is_contiguous()) or wf.dim() != 3 or out.dim() != 3:
        raise ValueError("wf [batch][na][na] and out [batch][nb][nb] must be contiguous CUDA tensors")
    batch, na, nb = int(wf.shape[0]), int(wf.shape[-1]), int(out.shape[-1])
    if wf.shape[1] != na or tuple(out.shape) != (batch, nb, nb):
        raise ValueError("wf must be [batch][na][na] and out [batch][nb][nb]")
    _, pi = _darr(pixel_in, batch)
    _, po = _darr(pixel_out, batch)
    _, lp = _darr(lam, batch)
    s = torch.cuda.current_stream(wf.device) if stream is None else stream
    st = lib().fresnel_mft_noalloc(ctypes.c_void_p(wf.data_ptr()), ctypes.c_void_p(out.data_ptr()), na, nb, batch,
                                   C128 if wf.dtype == torch.complex128 else C64, pi, po, lp, float(f), int(direction),
                                   ctypes.c_void_p(s.cuda_stream))
    if st != 0:
        raise FresnelError(st, "fresnel_mft_noalloc")


def run_surfaces(plan: Plan, wf, pixel, lam, surfaces: Sequence, maps=None) -> None:
    """Chain of fused surfaces ("10 optics ... 19 FFT"): one fresnel_surface_as per
    surface.  `maps[i]` = (amp, opd) device tensors or None for surface i."""
    for i, s in enumerate(surfaces):
        amp, opd = (maps[i] if maps is not None else (None, None))
        plan.surface_as(wf, pixel, lam, s.f, amp, opd, s.z)
