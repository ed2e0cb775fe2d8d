"""Thin ctypes binding of include/demag.h (argument marshalling only).

Function names follow the C ABI.  PyTorch is used for device memory and streams: tensors cross the
boundary as ``data_ptr()`` and the current CUDA stream as a raw handle.  There is no CPU fallback: if
the CUDA library is missing or fails, these calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdemag_b200.so")

DEMAG_FP32, DEMAG_FP64 = 0, 1
DEMAG_PBC_X, DEMAG_PBC_Y, DEMAG_PBC_Z = 1, 2, 4
STATUS = {0: "DEMAG_OK", 1: "DEMAG_ERR_INVALID_ARG", 2: "DEMAG_ERR_UNSUPPORTED", 3: "DEMAG_ERR_ALLOC",
          4: "DEMAG_ERR_CUDA", 5: "DEMAG_ERR_NO_KERNEL"}

EXPORTS = ["demag_plan_create", "demag_set_kernel", "demag_apply", "demag_energy", "demag_apply_atomistic",
           "demag_get_kernel_real", "demag_workspace_bytes", "demag_set_slab", "demag_launches_per_apply",
           "demag_last_error", "demag_plan_destroy", "demag_apply_profiled", "demag_path", "demag_apply_add"]


class DemagError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


_lib = None


def lib():
    """Load libdemag_b200.so (built by paper_2308_08447_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH) and os.environ.get("DEMAG_NO_AUTOBUILD") is None:
            try:                                   # build the CUDA extension in-tree (nvcc); still no CPU fallback
                from . import build as _build
                _build.build()
            except Exception:
                pass
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2308_08447_b200.build` "
                              "(the CUDA extension is required; there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i, d, u = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_uint
        L.demag_plan_create.argtypes = [ctypes.POINTER(vp), i, i, i, d, d, d, u, i]
        L.demag_set_kernel.argtypes = [vp, vp]
        L.demag_apply.argtypes = [vp, vp, vp, vp]
        L.demag_apply_add.argtypes = [vp, vp, vp, vp]
        L.demag_energy.argtypes = [vp, vp, vp, vp, vp]
        L.demag_apply_profiled.argtypes = [vp, vp, vp, vp, vp, vp]
        L.demag_apply_atomistic.argtypes = [vp, vp, vp, i, i, i, d, d, i, vp]
        L.demag_get_kernel_real.argtypes = [vp, vp]
        L.demag_workspace_bytes.argtypes = [vp]
        L.demag_workspace_bytes.restype = ctypes.c_size_t
        L.demag_set_slab.argtypes = [vp, i]
        L.demag_launches_per_apply.argtypes = [vp]
        L.demag_launches_per_apply.restype = i
        L.demag_path.argtypes = [vp]
        L.demag_path.restype = i
        L.demag_last_error.restype = ctypes.c_char_p
        L.demag_plan_destroy.argtypes = [vp]
        for name in EXPORTS:
            if name not in ("demag_workspace_bytes", "demag_launches_per_apply", "demag_last_error"):
                getattr(L, name).restype = i
        _lib = L
    return _lib


def _check(st: int):
    if st != 0:
        raise DemagError(st, lib().demag_last_error().decode())


def _stream(stream=None) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def demag_plan_create(nx, ny, nz, hx, hy, hz, pbc_flags=0, precision=DEMAG_FP32) -> int:
    h = ctypes.c_void_p()
    _check(lib().demag_plan_create(ctypes.byref(h), int(nx), int(ny), int(nz), float(hx), float(hy), float(hz),
                                   int(pbc_flags), int(precision)))
    return h.value


def demag_set_kernel(plan, N6_host=None):
    if N6_host is None:
        _check(lib().demag_set_kernel(plan, None))
        return
    a = np.ascontiguousarray(N6_host, dtype=np.float64)
    _check(lib().demag_set_kernel(plan, a.ctypes.data))


def demag_apply(plan, M, H, stream=None):
    _check(lib().demag_apply(plan, M.data_ptr(), H.data_ptr(), _stream(stream)))


def demag_apply_add(plan, M, Heff, stream=None):
    _check(lib().demag_apply_add(plan, M.data_ptr(), Heff.data_ptr(), _stream(stream)))


def demag_apply_profiled(plan, M, H, stream=None):
    """-> (stage_ms[5], stage_launches[5]) for x-R2C, y-fwd, z-fused, y-inv, x-C2R (synchronous)."""
    ms = (ctypes.c_float * 5)()
    cnt = (ctypes.c_int * 5)()
    _check(lib().demag_apply_profiled(plan, M.data_ptr(), H.data_ptr(), _stream(stream),
                                      ctypes.addressof(ms), ctypes.addressof(cnt)))
    return list(ms), list(cnt)


def demag_energy(plan, M, H, E, stream=None):
    _check(lib().demag_energy(plan, M.data_ptr(), H.data_ptr(), E.data_ptr(), _stream(stream)))


def demag_apply_atomistic(plan, S, Hs, c, mu_s, a, accumulate=False, stream=None):
    _check(lib().demag_apply_atomistic(plan, S.data_ptr(), Hs.data_ptr(), int(c[0]), int(c[1]), int(c[2]),
                                       float(mu_s), float(a), int(bool(accumulate)), _stream(stream)))


def demag_get_kernel_real(plan, n) -> np.ndarray:
    nx, ny, nz = n
    out = np.empty((6, nz, ny, nx), dtype=np.float64)
    _check(lib().demag_get_kernel_real(plan, out.ctypes.data))
    return out


def demag_workspace_bytes(plan) -> int:
    return int(lib().demag_workspace_bytes(plan))


def demag_set_slab(plan, kx_per_slab: int):
    _check(lib().demag_set_slab(plan, int(kx_per_slab)))


def demag_launches_per_apply(plan) -> int:
    return int(lib().demag_launches_per_apply(plan))


def demag_path(plan) -> int:
    return int(lib().demag_path(plan))


def demag_plan_destroy(plan):
    _check(lib().demag_plan_destroy(plan))


class Plan:
    """Context-managed plan handle (same calls as above, bound to one plan)."""

    def __init__(self, n, h, pbc_flags=0, precision=DEMAG_FP32):
        self.n, self.h, self.precision = tuple(n), tuple(h), precision
        self.handle = demag_plan_create(*n, *h, pbc_flags, precision)

    def set_kernel(self, N6_host=None):
        demag_set_kernel(self.handle, N6_host)
        return self

    def apply(self, M, H, stream=None):
        demag_apply(self.handle, M, H, stream)

    def apply_add(self, M, Heff, stream=None):
        demag_apply_add(self.handle, M, Heff, stream)

    def apply_profiled(self, M, H, stream=None):
        return demag_apply_profiled(self.handle, M, H, stream)

    def energy(self, M, H, E, stream=None):
        demag_energy(self.handle, M, H, E, stream)

    def apply_atomistic(self, S, Hs, c, mu_s, a, accumulate=False, stream=None):
        demag_apply_atomistic(self.handle, S, Hs, c, mu_s, a, accumulate, stream)

    def get_kernel_real(self):
        return demag_get_kernel_real(self.handle, self.n)

    def workspace_bytes(self):
        return demag_workspace_bytes(self.handle)

    def launches_per_apply(self):
        return demag_launches_per_apply(self.handle)

    def path(self):
        return demag_path(self.handle)

    def set_slab(self, k):
        demag_set_slab(self.handle, k)

    def close(self):
        if self.handle:
            demag_plan_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
