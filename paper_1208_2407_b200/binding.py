"""ctypes binding of libts.so -- argument marshalling only; every step of the path runs in the
CUDA kernels behind include/ts.h.  torch is used for device memory and stream handles."""
from __future__ import annotations

import ctypes
from pathlib import Path

TS_F32, TS_F64 = 0, 1
TS_CLOSED, TS_PERIODIC = 0, 1
TS_OK, TS_EINVAL, TS_EUNSUPPORTED, TS_EALLOC, TS_ECUDA = 0, 1, 2, 3, 4
TS_MAX_FUSE = 6

_LIB_PATH = Path(__file__).resolve().parent / "libts.so"
_lib = None

SYMBOLS = ["ts_plan_create", "ts_plan_create_xy", "ts_plan_create_3d", "ts_evolve", "ts_evolve_3d", "ts_evolve_u4", "ts_evolve_sep", "ts_evolve_tdep", "ts_slab_pass",
           "ts_norm", "ts_norm_static", "ts_evolve_host", "ts_plan_set_option",
           "ts_plan_get_info", "ts_u4_coefficients", "ts_plan_reserve", "ts_plan_get_launch_times", "ts_plan_destroy",
           "ts_last_error"]

# kinds reported by ts_plan_get_launch_times (include/ts.h)
LAUNCH_KINDS = {1: "per-sweep kernels", 2: "fused_kernel", 3: "stream_kernel", 4: "tiny_kernel",
                5: "line_kernel(rows)", 6: "line_kernel(columns)", 7: "xwin_kernel",
                8: "ycol_kernel", 9: "plane copies", 10: "expand_separable", 11: "line_kernel(z)",
                12: "phase_kernel"}


class TsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libts error {code}: {msg}")
        self.code = code


def lib():
    """Load libts.so; there is no fallback -- a missing library is an error."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_1208_2407_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(str(_LIB_PATH))
        vp, i64, dbl, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
        L.ts_plan_create.argtypes = [i64, i64, i32, i32]
        L.ts_plan_create.restype = vp
        L.ts_plan_create_xy.argtypes = [i64, i64, i32, i32, i32]
        L.ts_plan_create_xy.restype = vp
        L.ts_plan_create_3d.argtypes = [i64, i64, i64, i32, i32, i32, i32]
        L.ts_plan_create_3d.restype = vp
        L.ts_evolve.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, vp, i64, vp]
        L.ts_evolve.restype = i32
        L.ts_evolve_3d.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, vp, i64, vp]
        L.ts_evolve_3d.restype = i32
        L.ts_evolve_u4.argtypes = [vp, vp, vp, dbl, vp, vp, i64, vp]
        L.ts_evolve_u4.restype = i32
        L.ts_evolve_sep.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, vp, vp, i64, vp]
        L.ts_evolve_sep.restype = i32
        L.ts_evolve_tdep.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, ctypes.POINTER(vp), i64, vp]
        L.ts_evolve_tdep.restype = i32
        L.ts_slab_pass.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, vp, vp, i64,
                                   ctypes.POINTER(dbl), i32, vp, vp, i64, i64, i32, vp]
        L.ts_slab_pass.restype = i32
        L.ts_norm.argtypes = [vp, vp, vp, ctypes.POINTER(dbl), vp]
        L.ts_norm.restype = i32
        L.ts_norm_static.argtypes = [i32, vp, vp, i64, vp, vp]
        L.ts_norm_static.restype = i32
        L.ts_evolve_host.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, vp, i64]
        L.ts_evolve_host.restype = i32
        L.ts_plan_set_option.argtypes = [vp, ctypes.c_char_p, i64]
        L.ts_plan_set_option.restype = i32
        L.ts_plan_get_info.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(i64)]
        L.ts_plan_get_info.restype = i32
        L.ts_u4_coefficients.argtypes = [dbl, ctypes.POINTER(dbl)]
        L.ts_u4_coefficients.restype = i32
        L.ts_plan_reserve.argtypes = [vp, i32]
        L.ts_plan_reserve.restype = i32
        L.ts_plan_get_launch_times.argtypes = [vp, i32, ctypes.POINTER(i32),
                                               ctypes.POINTER(ctypes.c_float), ctypes.POINTER(i32)]
        L.ts_plan_get_launch_times.restype = i32
        L.ts_plan_destroy.argtypes = [vp]
        L.ts_plan_destroy.restype = i32
        L.ts_last_error.argtypes = []
        L.ts_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def last_error() -> str:
    return lib().ts_last_error().decode()


def _check(rc):
    if rc != TS_OK:
        raise TsError(rc, last_error())


def u4_coefficients(theta: float):
    """ts_u4_coefficients: the five (a_half, b_half, a_full, b_full) rows of one fourth-order step."""
    out = (ctypes.c_double * 20)()
    _check(lib().ts_u4_coefficients(float(theta), out))
    return [tuple(out[4 * k:4 * k + 4]) for k in range(5)]


def _dtype_code(torch_dtype):
    import torch
    if torch_dtype == torch.float32:
        return TS_F32
    if torch_dtype == torch.float64:
        return TS_F64
    raise TypeError("psi planes must be float32 or float64")


def _stream_handle(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def norm_static(psi_re, psi_im, out, stream=None) -> None:
    """ts_norm_static: sum |psi|^2 into the one-element float64 DEVICE tensor `out`, without any
    allocation and without a synchronisation (the partial sums live in a fixed 256 KB array of
    the library's device image; at most 2^29 sites; calls that overlap on the GPU race)."""
    import torch
    if not (psi_re.is_cuda and psi_im.is_cuda and out.is_cuda):
        raise ValueError("psi planes and out must be CUDA tensors")
    if psi_re.dtype != psi_im.dtype or psi_re.shape != psi_im.shape:
        raise ValueError("psi_re and psi_im must have the same dtype and shape")
    if not (psi_re.is_contiguous() and psi_im.is_contiguous()):
        raise ValueError("psi planes must be contiguous")
    if out.dtype != torch.float64 or out.numel() != 1:
        raise ValueError("out must be one float64 element")
    _check(lib().ts_norm_static(_dtype_code(psi_re.dtype), ctypes.c_void_p(psi_re.data_ptr()),
                                ctypes.c_void_p(psi_im.data_ptr()), int(psi_re.numel()),
                                ctypes.c_void_p(out.data_ptr()), _stream_handle(stream)))


class Plan:
    """ts_plan_create[_xy] / ts_plan_destroy.  boundary: "closed" or "periodic"; boundary_y
    defaults to the same (a different one per axis goes through ts_plan_create_xy)."""

    def __init__(self, nx: int, ny: int, dtype, boundary: str = "closed", boundary_y: str = None):
        self.nx, self.ny = int(nx), int(ny)
        self.dtype = dtype
        codes = {"closed": TS_CLOSED, "periodic": TS_PERIODIC}
        b = codes[boundary]
        if boundary_y is None:
            self._h = lib().ts_plan_create(self.nx, self.ny, _dtype_code(dtype), b)
        else:
            self._h = lib().ts_plan_create_xy(self.nx, self.ny, _dtype_code(dtype), b,
                                              codes[boundary_y])
        if not self._h:
            raise TsError(TS_EINVAL, last_error())

    def set_option(self, name: str, value: int):
        _check(lib().ts_plan_set_option(self._h, name.encode(), int(value)))

    def info(self, name: str) -> int:
        out = ctypes.c_int64(0)
        _check(lib().ts_plan_get_info(self._h, name.encode(), ctypes.byref(out)))
        return out.value

    def reserve(self, with_host_staging: int = 0):
        _check(lib().ts_plan_reserve(self._h, int(with_host_staging)))

    def launch_times(self):
        """[(kind, ms), ...] of the last evolve call (plan option "timing" = 1)."""
        n = ctypes.c_int(0)
        _check(lib().ts_plan_get_launch_times(self._h, 0, None, None, ctypes.byref(n)))
        if n.value == 0:
            return []
        kinds = (ctypes.c_int * n.value)()
        ms = (ctypes.c_float * n.value)()
        _check(lib().ts_plan_get_launch_times(self._h, n.value, kinds, ms, ctypes.byref(n)))
        return [(int(kinds[i]), float(ms[i])) for i in range(n.value)]

    def _planes(self, re, im):
        if re.dtype != self.dtype or im.dtype != self.dtype:
            raise TypeError("plane dtype differs from the plan's")
        if tuple(re.shape) != (self.ny, self.nx) or tuple(im.shape) != (self.ny, self.nx):
            raise ValueError("planes must have shape [ny][nx]")
        if not (re.is_contiguous() and im.is_contiguous()):
            raise ValueError("planes must be contiguous")

    def evolve(self, psi_re, psi_im, a_half, b_half, a_full, b_full, pot_phase=None,
               n_steps=1, stream=None):
        """ts_evolve on CUDA tensors, in place, asynchronous on `stream` (default: current)."""
        self._planes(psi_re, psi_im)
        if not (psi_re.is_cuda and psi_im.is_cuda):
            raise ValueError("evolve takes CUDA tensors; use evolve_host for host tensors")
        pot = None
        if pot_phase is not None:
            if pot_phase.dtype != self.dtype or tuple(pot_phase.shape) != (2, self.ny, self.nx) \
                    or not pot_phase.is_contiguous() or not pot_phase.is_cuda:
                raise ValueError("pot_phase must be a contiguous CUDA tensor [2][ny][nx]")
            pot = ctypes.c_void_p(pot_phase.data_ptr())
        _check(lib().ts_evolve(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                               ctypes.c_void_p(psi_im.data_ptr()), a_half, b_half, a_full, b_full,
                               pot, int(n_steps), _stream_handle(stream)))

    def _pot_ptr(self, pot_phase):
        if pot_phase is None:
            return None
        if pot_phase.dtype != self.dtype or tuple(pot_phase.shape) != (2, self.ny, self.nx) \
                or not pot_phase.is_contiguous() or not pot_phase.is_cuda:
            raise ValueError("pot_phase must be a contiguous CUDA tensor [2][ny][nx]")
        return ctypes.c_void_p(pot_phase.data_ptr())

    def evolve_u4(self, psi_re, psi_im, theta, pot_phase_p=None, pot_phase_q=None, n_steps=1,
                  stream=None):
        """ts_evolve_u4 (fourth-order step, Eq. 4) on CUDA tensors, in place, asynchronous."""
        self._planes(psi_re, psi_im)
        if not (psi_re.is_cuda and psi_im.is_cuda):
            raise ValueError("evolve_u4 takes CUDA tensors")
        _check(lib().ts_evolve_u4(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                                  ctypes.c_void_p(psi_im.data_ptr()), float(theta),
                                  self._pot_ptr(pot_phase_p), self._pot_ptr(pot_phase_q),
                                  int(n_steps), _stream_handle(stream)))

    def evolve_tdep(self, psi_re, psi_im, a_half, b_half, a_full, b_full, pot_phases, stream=None):
        """ts_evolve_tdep: one step per entry of pot_phases (CUDA tensors [2][ny][nx] or None)."""
        self._planes(psi_re, psi_im)
        n = len(pot_phases)
        arr = (ctypes.c_void_p * max(n, 1))()
        for k, t in enumerate(pot_phases):
            p = self._pot_ptr(t)
            arr[k] = p.value if p is not None else None
        _check(lib().ts_evolve_tdep(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                                    ctypes.c_void_p(psi_im.data_ptr()), a_half, b_half, a_full,
                                    b_full, arr, n, _stream_handle(stream)))

    def evolve_sep(self, psi_re, psi_im, a_half, b_half, a_full, b_full, phase_x, phase_y,
                   n_steps=1, stream=None):
        """ts_evolve_sep: separable potential phase, phase_x [2][nx], phase_y [2][ny] (CUDA)."""
        self._planes(psi_re, psi_im)
        for t, n in ((phase_x, self.nx), (phase_y, self.ny)):
            if t.dtype != self.dtype or tuple(t.shape) != (2, n) or not t.is_contiguous() \
                    or not t.is_cuda:
                raise ValueError("phase_x / phase_y must be contiguous CUDA tensors [2][n]")
        _check(lib().ts_evolve_sep(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                                   ctypes.c_void_p(psi_im.data_ptr()), a_half, b_half, a_full,
                                   b_full, ctypes.c_void_p(phase_x.data_ptr()),
                                   ctypes.c_void_p(phase_y.data_ptr()), int(n_steps),
                                   _stream_handle(stream)))

    def slab_pass(self, src, dst, up, dn, coef, phase_x=None, phase_y=None, y0=0, ny_global=0,
                  periodic_y_global=False, stream=None):
        """ts_slab_pass: src, dst = (re, im) CUDA planes of this slab; up, dn = (re, im) planes of
        the neighbours (any row count >= 2*n_sub; may be peer-GPU memory) or None at a closed edge;
        coef = sequence of (a_half, b_half, a_full, b_full), one per fused sub-step; phase_x
        [2][nx], phase_y [2][ny_global] = separable potential phase or None."""
        self._planes(src[0], src[1]); self._planes(dst[0], dst[1])

        def nb(t):
            if t is None:
                return None, None, 0
            re, im = t
            if re.dtype != self.dtype or re.shape[1] != self.nx or re.shape != im.shape or \
                    not (re.is_contiguous() and im.is_contiguous() and re.is_cuda):
                raise ValueError("neighbour planes must be contiguous CUDA tensors [rows][nx]")
            return ctypes.c_void_p(re.data_ptr()), ctypes.c_void_p(im.data_ptr()), re.shape[0]
        ur, ui, un = nb(up)
        dr, di, dn_rows = nb(dn)
        flat = [float(v) for row in coef for v in row]
        n_sub = len(flat) // 4
        table = (ctypes.c_double * len(flat))(*flat)
        px = py = None
        if phase_x is not None:
            if phase_x.dtype != self.dtype or tuple(phase_x.shape) != (2, self.nx) or \
                    phase_y.dtype != self.dtype or tuple(phase_y.shape) != (2, int(ny_global)) or \
                    not (phase_x.is_contiguous() and phase_y.is_contiguous() and phase_x.is_cuda):
                raise ValueError("phase_x [2][nx], phase_y [2][ny_global]: contiguous CUDA tensors")
            px, py = ctypes.c_void_p(phase_x.data_ptr()), ctypes.c_void_p(phase_y.data_ptr())
        _check(lib().ts_slab_pass(self._h, ctypes.c_void_p(src[0].data_ptr()),
                                  ctypes.c_void_p(src[1].data_ptr()),
                                  ctypes.c_void_p(dst[0].data_ptr()),
                                  ctypes.c_void_p(dst[1].data_ptr()), ur, ui, un, dr, di, dn_rows,
                                  table, n_sub, px, py, int(y0), int(ny_global),
                                  int(bool(periodic_y_global)), _stream_handle(stream)))

    def evolve_host(self, psi_re, psi_im, a_half, b_half, a_full, b_full, pot_phase=None,
                    n_steps=1):
        """ts_evolve_host on HOST tensors (pinned or pageable), in place, synchronous."""
        self._planes(psi_re, psi_im)
        if psi_re.is_cuda or psi_im.is_cuda:
            raise ValueError("evolve_host takes host tensors")
        pot = None
        if pot_phase is not None:
            if pot_phase.dtype != self.dtype or tuple(pot_phase.shape) != (2, self.ny, self.nx) \
                    or not pot_phase.is_contiguous() or pot_phase.is_cuda:
                raise ValueError("pot_phase must be a contiguous host tensor [2][ny][nx]")
            pot = ctypes.c_void_p(pot_phase.data_ptr())
        _check(lib().ts_evolve_host(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                                    ctypes.c_void_p(psi_im.data_ptr()), a_half, b_half, a_full,
                                    b_full, pot, int(n_steps)))

    def norm(self, psi_re, psi_im, stream=None) -> float:
        """ts_norm: sum |psi|^2 as a host float (synchronises the stream)."""
        self._planes(psi_re, psi_im)
        out = ctypes.c_double(0.0)
        _check(lib().ts_norm(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                             ctypes.c_void_p(psi_im.data_ptr()), ctypes.byref(out),
                             _stream_handle(stream)))
        return out.value

    def destroy(self):
        if self._h:
            lib().ts_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Plan3D(Plan):
    """ts_plan_create_3d: a lattice nx x ny x nz, planes [nz][ny][nx] (x fastest).  boundary: one
    name or a tuple (x, y, z) of "closed" / "periodic".  evolve = ts_evolve_3d; norm = ts_norm."""

    def __init__(self, nx: int, ny: int, nz: int, dtype, boundary="closed"):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.dtype = dtype
        codes = {"closed": TS_CLOSED, "periodic": TS_PERIODIC}
        b = (boundary,) * 3 if isinstance(boundary, str) else tuple(boundary)
        self._h = lib().ts_plan_create_3d(self.nx, self.ny, self.nz, _dtype_code(dtype),
                                          codes[b[0]], codes[b[1]], codes[b[2]])
        if not self._h:
            raise TsError(TS_EINVAL, last_error())

    def _planes(self, re, im):
        if re.dtype != self.dtype or im.dtype != self.dtype:
            raise TypeError("plane dtype differs from the plan's")
        shape = (self.nz, self.ny, self.nx)
        if tuple(re.shape) != shape or tuple(im.shape) != shape:
            raise ValueError(f"planes must have shape [nz][ny][nx] = {shape}")
        if not (re.is_contiguous() and im.is_contiguous()):
            raise ValueError("planes must be contiguous")

    def evolve(self, psi_re, psi_im, a_half, b_half, a_full, b_full, pot_phase=None,
               n_steps=1, stream=None):
        """ts_evolve_3d on CUDA tensors, in place, asynchronous on `stream` (default: current)."""
        self._planes(psi_re, psi_im)
        if not (psi_re.is_cuda and psi_im.is_cuda):
            raise ValueError("evolve takes CUDA tensors")
        pot = None
        if pot_phase is not None:
            if pot_phase.dtype != self.dtype or not pot_phase.is_contiguous() or not pot_phase.is_cuda \
                    or tuple(pot_phase.shape) != (2, self.nz, self.ny, self.nx):
                raise ValueError("pot_phase must be a contiguous CUDA tensor [2][nz][ny][nx]")
            pot = ctypes.c_void_p(pot_phase.data_ptr())
        _check(lib().ts_evolve_3d(self._h, ctypes.c_void_p(psi_re.data_ptr()),
                                  ctypes.c_void_p(psi_im.data_ptr()), a_half, b_half, a_full,
                                  b_full, pot, int(n_steps), _stream_handle(stream)))
