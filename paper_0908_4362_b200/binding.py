"""Thin ctypes binding of include/mhd.h -- argument marshalling only; every step of the hot path
runs in the CUDA kernels of libmhd.so.  There is NO CPU fallback: importing this module raises if
the library has not been built (``python -m paper_0908_4362_b200.build``).

The functions carry the names of the C ABI (``mhd_create``, ``mhd_set_state`` ...) and return the
status codes unchanged.  ``Solver`` is a small convenience wrapper around them that raises
``MHDError`` on failure and accepts numpy arrays or torch tensors (torch is used for device memory
and streams only).
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_longlong, c_size_t, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MHD_LIB") or os.path.join(_HERE, "libmhd.so")   # MHD_LIB: A/B-test another build of the same ABI

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build the CUDA library first (python -m paper_0908_4362_b200.build). "
        "This package has no CPU fallback."
    )

_lib = ctypes.CDLL(LIB_PATH)

MHD_F32, MHD_F64 = 0, 1
MHD_BC_PERIODIC, MHD_BC_OUTFLOW = 0, 1
MHD_HOST, MHD_DEVICE = 0, 1
MHD_OK, MHD_EINVAL, MHD_ENOMEM, MHD_ECUDA, MHD_ENONFINITE, MHD_ENOSTATE = 0, -1, -2, -3, -4, -5
MHD_OP_FLUID, MHD_OP_BPAIR, MHD_OP_SWEEP_FORWARD, MHD_OP_SWEEP_REVERSE, MHD_OP_MIDDLE_PAIR = 0, 1, 2, 3, 4

# every symbol include/mhd.h declares: (restype, argtypes)
_P8 = POINTER(c_void_p)
SIGNATURES = {
    "mhd_workspace_bytes": (c_size_t, [c_int, c_int, c_int, c_int]),
    "mhd_create": (c_int, [c_int, c_int, c_int, c_double, c_int, c_int, POINTER(c_void_p)]),
    "mhd_bind": (c_int, [c_void_p, c_void_p, c_size_t, c_void_p]),
    "mhd_destroy": (c_int, [c_void_p]),
    "mhd_set_state": (c_int, [c_void_p, _P8, c_int]),
    "mhd_get_state": (c_int, [c_void_p, _P8, c_int]),
    "mhd_cfl_dt": (c_int, [c_void_p, c_double, POINTER(c_double), POINTER(c_double)]),
    "mhd_step": (c_int, [c_void_p, c_int, c_double, POINTER(c_double)]),
    "mhd_step_fixed": (c_int, [c_void_p, c_int, c_double]),
    "mhd_run_until": (c_int, [c_void_p, c_double, c_double, c_longlong, POINTER(c_longlong), POINTER(c_double)]),
    "mhd_apply": (c_int, [c_void_p, c_int, c_int, c_int, c_double]),
    "mhd_get_step_index": (c_int, [c_void_p, POINTER(c_longlong)]),
    "mhd_set_step_index": (c_int, [c_void_p, c_longlong]),
    "mhd_get_time": (c_int, [c_void_p, POINTER(c_double)]),
    "mhd_diagnostics": (c_int, [c_void_p, POINTER(c_double), POINTER(c_double)]),
    "mhd_viz_range": (c_int, [c_void_p, c_int, POINTER(c_double), POINTER(c_double)]),
    "mhd_viz_curve": (c_int, [c_void_p, c_int, c_int, c_int, c_double, c_double, c_void_p]),
    "mhd_viz_slice": (c_int, [c_void_p, c_int, c_int, c_double, c_double, c_void_p, c_void_p]),
    "mhd_viz_volume": (c_int, [c_void_p, c_int, c_double, c_double, c_void_p, c_double, c_void_p]),
    "mhd_set_option": (c_int, [c_void_p, c_char_p, c_longlong]),
    "mhd_cmax_noalloc": (c_int, [_P8, c_int, c_int, c_int, c_double, c_int, c_int, c_void_p, c_void_p, c_char_p, c_size_t]),
    "mhd_launch_count": (c_longlong, [c_void_p]),
    "mhd_last_error": (c_char_p, [c_void_p]),
    "mhd_version": (c_char_p, []),
}
for _name, (_res, _args) in SIGNATURES.items():
    _fn = getattr(_lib, _name)          # AttributeError here = the library does not export the ABI
    _fn.restype, _fn.argtypes = _res, _args

mhd_workspace_bytes = _lib.mhd_workspace_bytes
mhd_create = _lib.mhd_create
mhd_bind = _lib.mhd_bind
mhd_destroy = _lib.mhd_destroy
mhd_set_state = _lib.mhd_set_state
mhd_get_state = _lib.mhd_get_state
mhd_cfl_dt = _lib.mhd_cfl_dt
mhd_step = _lib.mhd_step
mhd_step_fixed = _lib.mhd_step_fixed
mhd_run_until = _lib.mhd_run_until
mhd_viz_range = _lib.mhd_viz_range
mhd_viz_curve = _lib.mhd_viz_curve
mhd_viz_slice = _lib.mhd_viz_slice
mhd_viz_volume = _lib.mhd_viz_volume
MHD_VIZ_PRESSURE = 8
mhd_apply = _lib.mhd_apply
mhd_get_step_index = _lib.mhd_get_step_index
mhd_set_step_index = _lib.mhd_set_step_index
mhd_get_time = _lib.mhd_get_time
mhd_diagnostics = _lib.mhd_diagnostics
mhd_set_option = _lib.mhd_set_option
mhd_cmax_noalloc = _lib.mhd_cmax_noalloc
mhd_launch_count = _lib.mhd_launch_count
mhd_last_error = _lib.mhd_last_error
mhd_version = _lib.mhd_version


class MHDError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mhd error {code}: {msg}")
        self.code = code


def _is_torch(x):
    return type(x).__module__.startswith("torch")


class Solver:
    """One context.  Fields are lists of 8 arrays shaped (nz, ny, nx): numpy (host) or torch (host/cuda)."""

    def __init__(self, nx, ny, nz, gamma, precision="f32", bc=MHD_BC_PERIODIC, workspace=None, stream=None):
        self.prec = {"f32": MHD_F32, "f64": MHD_F64, MHD_F32: MHD_F32, MHD_F64: MHD_F64}[precision]
        self.shape = (nz, ny, nx)
        self.np_dtype = np.float32 if self.prec == MHD_F32 else np.float64
        self._h = c_void_p()
        rc = mhd_create(nx, ny, nz, float(gamma), self.prec, int(bc), byref(self._h))
        if rc:
            raise MHDError(rc, mhd_last_error(None).decode())
        self._keep = workspace
        if workspace is not None or stream is not None:
            ptr = workspace.data_ptr() if workspace is not None else None
            nbytes = workspace.numel() * workspace.element_size() if workspace is not None else 0
            sptr = getattr(stream, "cuda_stream", stream)
            self._check(mhd_bind(self._h, ptr, nbytes, sptr))

    def _check(self, rc):
        if rc:
            raise MHDError(rc, mhd_last_error(self._h).decode())

    def close(self):
        if self._h:
            mhd_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptrs(self, fields):
        if len(fields) != 8:
            raise ValueError("need 8 fields")
        ptrs, where = [], None
        for f in fields:
            if _is_torch(f):
                import torch
                want = torch.float32 if self.prec == MHD_F32 else torch.float64
                if f.dtype != want or not f.is_contiguous() or tuple(f.shape) != self.shape:
                    raise ValueError("field has wrong dtype/shape or is not contiguous")
                w = MHD_DEVICE if f.is_cuda else MHD_HOST
                ptrs.append(f.data_ptr())
            else:
                if f.dtype != self.np_dtype or not f.flags.c_contiguous or f.shape != self.shape:
                    raise ValueError("field has wrong dtype/shape or is not contiguous")
                w = MHD_HOST
                ptrs.append(f.ctypes.data)
            if where is None:
                where = w
            elif where != w:
                raise ValueError("all fields must live on the same side")
        return (c_void_p * 8)(*ptrs), where

    def set_state(self, fields):
        p, where = self._ptrs(fields)
        self._check(mhd_set_state(self._h, p, where))

    def get_state(self, out=None):
        if out is None:
            out = [np.empty(self.shape, self.np_dtype) for _ in range(8)]
        p, where = self._ptrs(out)
        self._check(mhd_get_state(self._h, p, where))
        return out

    def cfl_dt(self, cfl):
        dt, cm = c_double(), c_double()
        self._check(mhd_cfl_dt(self._h, float(cfl), byref(dt), byref(cm)))
        return dt.value, cm.value

    def step(self, n, cfl, sync=True):
        if sync:
            t = c_double()
            self._check(mhd_step(self._h, int(n), float(cfl), byref(t)))
            return t.value
        self._check(mhd_step(self._h, int(n), float(cfl), None))
        return None

    def step_fixed(self, n, dt):
        self._check(mhd_step_fixed(self._h, int(n), float(dt)))

    def run_until(self, t_end, cfl, max_steps=1 << 40):
        """-> (steps taken, time reached); the stop test and the last-step clipping run on the device"""
        n, t = c_longlong(), c_double()
        self._check(mhd_run_until(self._h, float(t_end), float(cfl), int(max_steps), byref(n), byref(t)))
        return n.value, t.value

    def apply(self, op, d, reverse, dt):
        self._check(mhd_apply(self._h, int(op), int(d), int(bool(reverse)), float(dt)))

    @property
    def step_index(self):
        s = c_longlong()
        self._check(mhd_get_step_index(self._h, byref(s)))
        return s.value

    @step_index.setter
    def step_index(self, s):
        self._check(mhd_set_step_index(self._h, int(s)))

    def time(self):
        t = c_double()
        self._check(mhd_get_time(self._h, byref(t)))
        return t.value

    def diagnostics(self):
        sums = (c_double * 8)()
        dv = c_double()
        self._check(mhd_diagnostics(self._h, sums, byref(dv)))
        return list(sums), dv.value

    # ---- headless visualisation stage: device buffers (torch tensors or raw device pointers) in, nothing copied ----
    @staticmethod
    def _dev(x):
        return x.data_ptr() if _is_torch(x) else int(x)

    def viz_range(self, field):
        lo, hi = c_double(), c_double()
        self._check(mhd_viz_range(self._h, int(field), byref(lo), byref(hi)))
        return lo.value, hi.value

    def viz_curve(self, field, j, k, vmin, vmax, xy):
        self._check(mhd_viz_curve(self._h, int(field), int(j), int(k), float(vmin), float(vmax), self._dev(xy)))

    def viz_slice(self, field, k, vmin, vmax, lut, rgba):
        self._check(mhd_viz_slice(self._h, int(field), int(k), float(vmin), float(vmax), self._dev(lut), self._dev(rgba)))

    def viz_volume(self, field, vmin, vmax, lut, opacity, rgba):
        self._check(mhd_viz_volume(self._h, int(field), float(vmin), float(vmax), self._dev(lut), float(opacity), self._dev(rgba)))

    def set_option(self, key, value):
        self._check(mhd_set_option(self._h, key.encode(), int(value)))

    def launch_count(self):
        return int(mhd_launch_count(self._h))
