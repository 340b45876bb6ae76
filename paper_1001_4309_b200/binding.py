"""ctypes binding of ``libsfd.so`` — argument marshalling only; every step of the hot path runs in
the library's CUDA kernels.  Names mirror ``include/sfd.h``.

PyTorch appears here only as the owner of device memory and streams: tensors are passed down as
``data_ptr()`` and the stream as ``torch.cuda.current_stream().cuda_stream``.

There is no CPU fallback: importing this module raises if ``libsfd.so`` is missing, and every call
raises ``SfdError`` on a non-zero return code."""
from __future__ import annotations

import ctypes as C
import pathlib
import re

import numpy as np

_PKG = pathlib.Path(__file__).resolve().parent
LIB_PATH = _PKG / "libsfd.so"        # the in-tree build, nothing else
HEADER_PATH = _PKG.parent / "include" / "sfd.h"

SFD_OK, SFD_EINVAL, SFD_ENOMEM, SFD_ECUDA, SFD_EUNSUPPORTED = 0, -1, -2, -3, -4
SFD_U8, SFD_F32, SFD_C64 = 0, 1, 2
SFD_KERNELS_AUTO, SFD_KERNELS_GENERIC = 0, 1

if not LIB_PATH.exists():
    raise ImportError(
        f"{LIB_PATH} is not built — run `python -m paper_1001_4309_b200.build` (needs nvcc). "
        "There is no CPU fallback for the Shifted-Fresnel hot path.")

_lib = C.CDLL(str(LIB_PATH))

_dp = C.POINTER(C.c_double)
_vp = C.c_void_p
_sig = {
    "sfd_plan_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_double, _dp, _dp, _dp, _dp,
                                  _dp, C.c_int]),
    "sfd_plan_create_general": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_double] + [_dp] * 9
                                + [C.c_int]),
    "sfd_plan_update_view_general": (C.c_int, [_vp, C.c_int] + [C.c_double] * 9),
    "sfd_plan_create_rect": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double] + [_dp] * 9
                             + [C.c_int]),
    "sfd_plan_set_input_window": (C.c_int, [_vp, C.c_longlong, C.c_int, C.c_int]),
    "sfd_plan_update_view_async": (C.c_int, [_vp, C.c_int] + [C.c_double] * 5 + [_vp]),
    "sfd_plan_update_view_general_async": (C.c_int, [_vp, C.c_int] + [C.c_double] * 9 + [_vp]),
    "sfd_plan_last_update_host_ms": (C.c_double, [_vp]),
    "sfd_plan_get_nx": (C.c_int, [_vp]),
    "sfd_plan_get_ny": (C.c_int, [_vp]),
    "sfd_plan_get_device": (C.c_int, [_vp]),
    "sfd_host_dft32": (C.c_int, [C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_int, C.c_int]),
    "sfd_measure_pipes": (C.c_int, [_dp]),
    "sfd_measure_memory_pipes": (C.c_int, [_dp]),
    "sfd_asm_plan_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                      C.c_double, _dp, C.c_int, C.c_int]),
    "sfd_asm_execute": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "sfd_asm_plan_destroy": (C.c_int, [_vp]),
    "sfd_asm_plan_device_bytes": (C.c_longlong, [_vp]),
    "sfd_asm_last_cuda_error": (C.c_char_p, []),
    "sfd_host_tables_general": (C.c_int, [C.c_int] + [C.c_double] * 6 + [_dp, _dp, _dp]),
    "sfd_execute": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "sfd_execute_u8": (C.c_int, [_vp, _vp, _vp, _vp]),
    "sfd_execute_focus": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "sfd_quantise_u8_static": (C.c_int, [_vp, C.c_int, C.c_longlong, _vp, _vp]),
    "sfd_static_max_views": (C.c_int, []),
    "sfd_static_last_error": (C.c_char_p, []),
    "sfd_stream_run": (C.c_int, [_vp, _vp, C.c_int, _vp, _dp]),
    "sfd_plan_update_view": (C.c_int, [_vp, C.c_int] + [C.c_double] * 5),
    "sfd_plan_destroy": (C.c_int, [_vp]),
    "sfd_plan_get_n": (C.c_int, [_vp]),
    "sfd_plan_get_views": (C.c_int, [_vp]),
    "sfd_plan_get_m": (C.c_int, [_vp]),
    "sfd_plan_device_bytes": (C.c_longlong, [_vp]),
    "sfd_plan_select_kernels": (C.c_int, [_vp, C.c_int]),
    "sfd_plan_uses_warp_kernels": (C.c_int, [_vp]),
    "sfd_plan_set_timing": (C.c_int, [_vp, C.c_int]),
    "sfd_plan_last_kernel_ms": (C.c_int, [_vp, C.POINTER(C.c_float)]),
    "sfd_launch_count": (C.c_longlong, []),
    "sfd_host_tables": (C.c_int, [C.c_int] + [C.c_double] * 5 + [_dp, _dp, _dp]),
    "sfd_error_string": (C.c_char_p, [C.c_int]),
    "sfd_last_cuda_error": (C.c_char_p, []),
    "sfd_version": (C.c_char_p, []),
}
for _name, (_res, _args) in _sig.items():
    _f = getattr(_lib, _name)          # AttributeError here = the library lacks a declared symbol
    _f.restype, _f.argtypes = _res, _args


def declared_symbols():
    """Names of all functions ``include/sfd.h`` declares (parsed from the header)."""
    text = HEADER_PATH.read_text()
    return sorted(set(re.findall(r"SFD_API[^;(]*?\b(sfd_\w+)\s*\(", text)))


class SfdError(RuntimeError):
    def __init__(self, code, where):
        msg = _lib.sfd_error_string(code).decode()
        if code == SFD_ECUDA:
            msg += ": " + _lib.sfd_last_cuda_error().decode()
        super().__init__(f"{where} failed with {code} ({msg})")
        self.code = code


def _chk(code, where):
    if code != SFD_OK:
        raise SfdError(code, where)


def _darr(v, n=None):
    a = np.ascontiguousarray(np.atleast_1d(np.asarray(v, dtype=np.float64)))
    if n is not None and n >= 1 and a.shape != (n,):      # the C side reads n values
        raise ValueError(f"expected {n} per-view values, got shape {a.shape}")
    return a


def _ptr(t):
    """Device/host address of a torch tensor, a numpy array, an int, or None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


# ---- functions with the names of the C ABI -------------------------------------------------------
def sfd_version():
    return _lib.sfd_version().decode()


def sfd_error_string(code):
    return _lib.sfd_error_string(int(code)).decode()


def sfd_last_cuda_error():
    return _lib.sfd_last_cuda_error().decode()


def sfd_launch_count():
    return int(_lib.sfd_launch_count())


def sfd_plan_create(N, n_views, lam, p1, p2, z, Ox, Oy, in_dtype=SFD_U8):
    """Returns the opaque plan handle (an int).  Per-view arrays are host sequences of floats."""
    arrs = [_darr(a, n_views) for a in (p1, p2, z, Ox, Oy)]
    h = _vp()
    _chk(_lib.sfd_plan_create(C.byref(h), int(N), int(n_views), float(lam),
                              *[a.ctypes.data_as(_dp) for a in arrs], int(in_dtype)),
         "sfd_plan_create")
    return h.value


def sfd_plan_create_general(N, n_views, lam, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y,
                            in_dtype=SFD_U8):
    """General geometry: separate x/y pitches and hologram-window offsets (include/sfd.h)."""
    arrs = [_darr(a, n_views) for a in (p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y)]
    h = _vp()
    _chk(_lib.sfd_plan_create_general(C.byref(h), int(N), int(n_views), float(lam),
                                      *[a.ctypes.data_as(_dp) for a in arrs], int(in_dtype)),
         "sfd_plan_create_general")
    return h.value


def sfd_plan_create_rect(Nx, Ny, n_views, lam, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y,
                         in_dtype=SFD_U8):
    """Rectangular grid [Ny][Nx] with the general geometry (include/sfd.h)."""
    arrs = [_darr(a, n_views) for a in (p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y)]
    h = _vp()
    _chk(_lib.sfd_plan_create_rect(C.byref(h), int(Nx), int(Ny), int(n_views), float(lam),
                                   *[a.ctypes.data_as(_dp) for a in arrs], int(in_dtype)),
         "sfd_plan_create_rect")
    return h.value


def sfd_plan_set_input_window(plan, row_stride, row0, col0):
    _chk(_lib.sfd_plan_set_input_window(plan, int(row_stride), int(row0), int(col0)),
         "sfd_plan_set_input_window")


def sfd_plan_update_view_async(plan, view, p1, p2, z, Ox, Oy, stream=None):
    _chk(_lib.sfd_plan_update_view_async(plan, int(view), float(p1), float(p2), float(z), float(Ox),
                                         float(Oy), _stream(stream)), "sfd_plan_update_view_async")


def sfd_plan_update_view_general_async(plan, view, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y,
                                       stream=None):
    _chk(_lib.sfd_plan_update_view_general_async(
        plan, int(view), *map(float, (p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y)), _stream(stream)),
        "sfd_plan_update_view_general_async")


def sfd_plan_last_update_host_ms(plan):
    return float(_lib.sfd_plan_last_update_host_ms(plan))


def sfd_plan_get_nx(plan):
    return int(_lib.sfd_plan_get_nx(plan))


def sfd_plan_get_ny(plan):
    return int(_lib.sfd_plan_get_ny(plan))


def sfd_plan_get_device(plan):
    return int(_lib.sfd_plan_get_device(plan))


def sfd_host_dft32(x, lane=0, twiddled=False):
    """Host-only: one radix-32 stage of the warp FFT stepped on the CPU; x = 32 complex values."""
    a = np.ascontiguousarray(np.asarray(x, dtype=np.complex64)).view(np.float32)
    if a.shape != (64,):
        raise ValueError("expected 32 complex values")
    out = np.empty(64, np.float32)
    fp = C.POINTER(C.c_float)
    _chk(_lib.sfd_host_dft32(a.ctypes.data_as(fp), out.ctypes.data_as(fp), int(lane),
                             int(bool(twiddled))), "sfd_host_dft32")
    return out.view(np.complex64)


def sfd_measure_pipes():
    """(fp32 FMA TFLOP/s, cycles per stage-A butterfly, cycles per stage-B butterfly, SM GHz)."""
    out = np.zeros(4, np.float64)
    _chk(_lib.sfd_measure_pipes(out.ctypes.data_as(_dp)), "sfd_measure_pipes")
    return tuple(float(v) for v in out)


def sfd_measure_memory_pipes():
    """(shared memory B/clk/SM in the transposes' access pattern, tensor-memory load B/clk/sub-partition with
    one warp, with two warps per sub-partition, cycles of a dependent tcgen05.ld)."""
    out = np.zeros(4, np.float64)
    _chk(_lib.sfd_measure_memory_pipes(out.ctypes.data_as(_dp)), "sfd_measure_memory_pipes")
    return tuple(float(v) for v in out)


def sfd_plan_update_view_general(plan, view, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y):
    _chk(_lib.sfd_plan_update_view_general(plan, int(view), *map(float, (p1x, p1y, p2x, p2y, z, O0x,
                                                                         O0y, O1x, O1y))),
         "sfd_plan_update_view_general")


def sfd_execute(plan, hologram_dev, field_dev, intensity_dev, stream=None):
    _chk(_lib.sfd_execute(plan, _ptr(hologram_dev), _ptr(field_dev), _ptr(intensity_dev),
                          _stream(stream)), "sfd_execute")


def sfd_quantise_u8_static(intensity_dev, n_views, pixels_per_view, intensity_u8_dev, stream=None):
    code = _lib.sfd_quantise_u8_static(_ptr(intensity_dev), n_views, pixels_per_view, _ptr(intensity_u8_dev),
                                       _stream(stream))
    if code != SFD_OK:
        err = SfdError(code, "sfd_quantise_u8_static")
        err.args = (err.args[0] + ": " + _lib.sfd_static_last_error().decode(),)
        raise err


def sfd_static_max_views():
    return int(_lib.sfd_static_max_views())


def sfd_static_last_error():
    return _lib.sfd_static_last_error().decode()


def sfd_execute_focus(plan, hologram_dev, moments_dev, intensity_dev=None, stream=None):
    _chk(_lib.sfd_execute_focus(plan, _ptr(hologram_dev), _ptr(moments_dev), _ptr(intensity_dev),
                                _stream(stream)), "sfd_execute_focus")


def sfd_execute_u8(plan, hologram_dev, intensity_u8_dev, stream=None):
    _chk(_lib.sfd_execute_u8(plan, _ptr(hologram_dev), _ptr(intensity_u8_dev), _stream(stream)),
         "sfd_execute_u8")


def sfd_stream_run(plan, holograms_pinned, n_frames, out_pinned):
    """Returns the device-measured seconds from first H2D to last D2H."""
    sec = C.c_double(0.0)
    _chk(_lib.sfd_stream_run(plan, _ptr(holograms_pinned), int(n_frames), _ptr(out_pinned),
                             C.byref(sec)), "sfd_stream_run")
    return sec.value


def sfd_plan_update_view(plan, view, p1, p2, z, Ox, Oy):
    _chk(_lib.sfd_plan_update_view(plan, int(view), float(p1), float(p2), float(z), float(Ox),
                                   float(Oy)), "sfd_plan_update_view")


def sfd_plan_destroy(plan):
    _chk(_lib.sfd_plan_destroy(plan), "sfd_plan_destroy")


def sfd_plan_get_n(plan):
    return int(_lib.sfd_plan_get_n(plan))


def sfd_plan_get_views(plan):
    return int(_lib.sfd_plan_get_views(plan))


def sfd_plan_get_m(plan):
    return int(_lib.sfd_plan_get_m(plan))


def sfd_plan_device_bytes(plan):
    return int(_lib.sfd_plan_device_bytes(plan))


def sfd_plan_select_kernels(plan, which):
    _chk(_lib.sfd_plan_select_kernels(plan, int(which)), "sfd_plan_select_kernels")


def sfd_plan_uses_warp_kernels(plan):
    return int(_lib.sfd_plan_uses_warp_kernels(plan))


def sfd_plan_set_timing(plan, enable):
    _chk(_lib.sfd_plan_set_timing(plan, int(bool(enable))), "sfd_plan_set_timing")


def sfd_plan_last_kernel_ms(plan):
    ms = (C.c_float * 3)()
    _chk(_lib.sfd_plan_last_kernel_ms(plan, ms), "sfd_plan_last_kernel_ms")
    return [float(x) for x in ms]


def sfd_host_tables(N, lam, p1, p2, z, off):
    """Host-only: (pre[N], post[N], H[2N]) complex128, one axis of one view (see sfd.h)."""
    pre = np.empty(N, np.complex128)
    post = np.empty(N, np.complex128)
    H = np.empty(2 * N, np.complex128)
    _chk(_lib.sfd_host_tables(int(N), float(lam), float(p1), float(p2), float(z), float(off),
                              pre.ctypes.data_as(_dp), post.ctypes.data_as(_dp),
                              H.ctypes.data_as(_dp)), "sfd_host_tables")
    return pre, post, H


def sfd_host_tables_general(N, lam, p1, p2, z, off0, off):
    """The same with the hologram window shifted by ``off0`` along the axis."""
    pre = np.empty(N, np.complex128)
    post = np.empty(N, np.complex128)
    H = np.empty(2 * N, np.complex128)
    _chk(_lib.sfd_host_tables_general(int(N), float(lam), float(p1), float(p2), float(z),
                                      float(off0), float(off), pre.ctypes.data_as(_dp),
                                      post.ctypes.data_as(_dp), H.ctypes.data_as(_dp)),
         "sfd_host_tables_general")
    return pre, post, H


def sfd_asm_plan_create(Nx, Ny, n_planes, lam, px, py, z, in_dtype=SFD_C64, band_limit=False):
    """Angular-spectrum plan (include/sfd.h); returns the opaque handle."""
    zz = _darr(z, n_planes)
    h = _vp()
    code = _lib.sfd_asm_plan_create(C.byref(h), int(Nx), int(Ny), int(n_planes), float(lam), float(px),
                                    float(py), zz.ctypes.data_as(_dp), int(in_dtype), int(bool(band_limit)))
    if code == SFD_ECUDA:
        raise SfdError(code, "sfd_asm_plan_create: " + _lib.sfd_asm_last_cuda_error().decode())
    _chk(code, "sfd_asm_plan_create")
    return h.value


def sfd_asm_execute(plan, u0_dev, field_dev, intensity_dev, phase_dev, stream=None):
    code = _lib.sfd_asm_execute(plan, _ptr(u0_dev), _ptr(field_dev), _ptr(intensity_dev),
                                _ptr(phase_dev), _stream(stream))
    if code == SFD_ECUDA:
        raise SfdError(code, "sfd_asm_execute: " + _lib.sfd_asm_last_cuda_error().decode())
    _chk(code, "sfd_asm_execute")


def sfd_asm_plan_destroy(plan):
    _chk(_lib.sfd_asm_plan_destroy(plan), "sfd_asm_plan_destroy")


def sfd_asm_plan_device_bytes(plan):
    return int(_lib.sfd_asm_plan_device_bytes(plan))


def sfd_asm_last_cuda_error():
    return _lib.sfd_asm_last_cuda_error().decode()


class AsmPlan:
    """Angular-spectrum plan: ``AsmPlan(Nx, Ny, lam, pitch, z=[...], in_dtype=SFD_C64, band_limit=False)``;
    ``pitch`` a scalar or ``(px, py)``.  Allocation of outputs is the only thing it adds."""

    def __init__(self, Nx, Ny, lam, pitch, z, in_dtype=SFD_C64, band_limit=False):
        px, py = (pitch, pitch) if np.ndim(pitch) == 0 else pitch
        self.Nx, self.Ny, self.P, self.in_dtype = int(Nx), int(Ny), len(np.atleast_1d(z)), int(in_dtype)
        self.handle = sfd_asm_plan_create(Nx, Ny, self.P, lam, px, py, z, in_dtype, band_limit)

    def close(self):
        if self.handle:
            sfd_asm_plan_destroy(self.handle)
            self.handle = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def execute(self, u0, field=True, intensity=True, phase=True, stream=None):
        """Returns ``(field complex64, intensity float32, phase float32)``, each ``[P, Ny, Nx]`` or None."""
        import torch
        want = torch.float32 if self.in_dtype == SFD_F32 else torch.complex64
        if (u0.dtype != want or tuple(u0.shape) != (self.Ny, self.Nx) or not u0.is_cuda
                or not u0.is_contiguous()):
            raise ValueError(f"input must be a contiguous CUDA tensor [{self.Ny},{self.Nx}] {want}")
        shape = (self.P, self.Ny, self.Nx)
        f = torch.empty(shape, dtype=torch.complex64, device=u0.device) if field else None
        I = torch.empty(shape, dtype=torch.float32, device=u0.device) if intensity else None
        ph = torch.empty(shape, dtype=torch.float32, device=u0.device) if phase else None
        sfd_asm_execute(self.handle, u0, f, I, ph, stream)
        return f, I, ph

    @property
    def device_bytes(self):
        return sfd_asm_plan_device_bytes(self.handle)


# ---- convenience wrapper: owns the handle, allocates outputs with torch --------------------------
class Plan:
    """``Plan(workload)`` or ``Plan(N=..., lam=..., p1=..., p2=..., z=..., Ox=..., Oy=...,
    in_dtype=...)``; a context manager.  Allocation of outputs is the only thing it adds."""

    def __init__(self, workload=None, **kw):
        if workload is not None:
            kw = dict(N=workload.N, lam=workload.lam, p1=workload.p1, p2=workload.p2,
                      z=workload.z, Ox=workload.Ox, Oy=workload.Oy, in_dtype=workload.in_dtype)
        self.Nx = int(kw["Nx"] if "Nx" in kw else kw["N"])
        self.Ny = int(kw["Ny"] if "Ny" in kw else kw["N"])
        self.N = self.Nx
        self.V = len(np.atleast_1d(kw["z"]))
        self.in_dtype = int(kw.get("in_dtype", SFD_U8))
        self.frame_shape = None      # set by set_input_window: hologram tensors are whole frames
        if "Nx" in kw:      # rectangular grid [Ny][Nx], general geometry
            self.handle = sfd_plan_create_rect(
                self.Nx, self.Ny, self.V, kw["lam"], kw["p1x"], kw["p1y"], kw["p2x"], kw["p2y"],
                kw["z"], kw["O0x"], kw["O0y"], kw["O1x"], kw["O1y"], self.in_dtype)
        elif "p1x" in kw:   # general geometry: p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y
            self.handle = sfd_plan_create_general(
                self.N, self.V, kw["lam"], kw["p1x"], kw["p1y"], kw["p2x"], kw["p2y"], kw["z"],
                kw["O0x"], kw["O0y"], kw["O1x"], kw["O1y"], self.in_dtype)
        else:
            self.handle = sfd_plan_create(self.N, self.V, kw["lam"], kw["p1"], kw["p2"], kw["z"],
                                          kw["Ox"], kw["Oy"], self.in_dtype)

    def close(self):
        if self.handle:
            sfd_plan_destroy(self.handle)
            self.handle = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check_holo(self, hologram):
        import torch
        want = torch.uint8 if self.in_dtype == SFD_U8 else torch.float32
        shape = self.frame_shape or (self.Ny, self.Nx)
        if (hologram.dtype != want or tuple(hologram.shape) != shape
                or not hologram.is_cuda or not hologram.is_contiguous()):
            raise ValueError(f"hologram must be a contiguous CUDA tensor {list(shape)} {want}")

    def set_input_window(self, frame_shape, row0, col0):
        """Holograms passed to execute* are whole frames ``frame_shape = (rows, row_stride)``; the
        plan reads its Ny x Nx window at (row0, col0) in place.  ``frame_shape=None`` = dense."""
        if frame_shape is None:
            sfd_plan_set_input_window(self.handle, 0, 0, 0)
            self.frame_shape = None
            return
        rows, stride = int(frame_shape[0]), int(frame_shape[1])
        if row0 + self.Ny > rows:
            raise ValueError("window exceeds the frame")
        sfd_plan_set_input_window(self.handle, stride, row0, col0)
        self.frame_shape = (rows, stride)

    def execute(self, hologram, field=True, intensity=True, stream=None):
        """Returns ``(field complex64 [V,N,N] | None, intensity float32 [V,N,N] | None)``.
        ``field`` / ``intensity`` may be ``True`` (allocate), ``False`` (skip) or a tensor."""
        import torch
        self._check_holo(hologram)
        shape = (self.V, self.Ny, self.Nx)
        if field is True:
            field = torch.empty(shape, dtype=torch.complex64, device=hologram.device)
        elif field is False:
            field = None
        if intensity is True:
            intensity = torch.empty(shape, dtype=torch.float32, device=hologram.device)
        elif intensity is False:
            intensity = None
        sfd_execute(self.handle, hologram, field, intensity, stream)
        return field, intensity

    def execute_focus(self, hologram, intensity=False, stream=None):
        """Depth stack / focus sweep: returns ``(moments[V, 2] float64 = (sum I, sum I^2),
        intensity[V, N, N] or None)`` as device tensors."""
        import torch
        self._check_holo(hologram)
        mom = torch.empty((self.V, 2), dtype=torch.float64, device=hologram.device)
        I = (torch.empty((self.V, self.Ny, self.Nx), dtype=torch.float32, device=hologram.device)
             if intensity else None)
        sfd_execute_focus(self.handle, hologram, mom, I, stream)
        return mom, I

    def execute_u8(self, hologram, out=None, stream=None):
        import torch
        self._check_holo(hologram)
        if out is None:
            out = torch.empty((self.V, self.Ny, self.Nx), dtype=torch.uint8, device=hologram.device)
        sfd_execute_u8(self.handle, hologram, out, stream)
        return out

    def stream_run(self, holograms_pinned, out_pinned=None):
        """``holograms_pinned``: pinned CPU tensor [F,N,N]; returns ``(out [F,V,N,N] uint8 pinned,
        seconds)``."""
        import torch
        F = int(holograms_pinned.shape[0])
        if not holograms_pinned.is_pinned() or not holograms_pinned.is_contiguous():
            raise ValueError("holograms must be a contiguous pinned CPU tensor")
        if out_pinned is None:
            out_pinned = torch.empty((F, self.V, self.Ny, self.Nx), dtype=torch.uint8).pin_memory()
        sec = sfd_stream_run(self.handle, holograms_pinned, F, out_pinned)
        return out_pinned, sec

    def update_view_general(self, view, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y):
        sfd_plan_update_view_general(self.handle, view, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y)

    def update_view(self, view, p1, p2, z, Ox, Oy):
        sfd_plan_update_view(self.handle, view, p1, p2, z, Ox, Oy)

    def update_view_async(self, view, p1, p2, z, Ox, Oy, stream=None):
        sfd_plan_update_view_async(self.handle, view, p1, p2, z, Ox, Oy, stream)

    @property
    def last_update_host_ms(self):
        return sfd_plan_last_update_host_ms(self.handle)

    def select_kernels(self, which):
        sfd_plan_select_kernels(self.handle, which)

    @property
    def uses_warp_kernels(self):
        """True when both passes run the warp-per-branch kernels (bit 0 = pass y, bit 1 = pass x)."""
        return sfd_plan_uses_warp_kernels(self.handle) == 3

    @property
    def warp_kernel_mask(self):
        return sfd_plan_uses_warp_kernels(self.handle)

    def set_timing(self, enable=True):
        sfd_plan_set_timing(self.handle, enable)

    def last_kernel_ms(self):
        return sfd_plan_last_kernel_ms(self.handle)

    @property
    def device_bytes(self):
        return sfd_plan_device_bytes(self.handle)
