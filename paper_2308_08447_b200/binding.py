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
           "demag_last_error", "demag_plan_destroy", "demag_apply_profiled", "demag_path", "demag_apply_add",
           "demag_shard_range", "demag_plan_create_sharded", "demag_shard_info", "demag_shard_buffers",
           "demag_shard_ipc_export", "demag_shard_ipc_connect", "demag_shard_set_peers", "demag_apply_sharded",
           "demag_set_pbc_images", "demag_extrapolate", "demag_atomistic_reserve",
           "demag_apply_atomistic_static", "demag_static_scratch_bytes",
           "demag_plan_dims", "demag_llg_create", "demag_llg_set_field", "demag_llg_step", "demag_llg_mean",
           "demag_llg_counts", "demag_llg_reset", "demag_llg_destroy"]


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
        L.demag_atomistic_reserve.argtypes = [vp]
        L.demag_apply_atomistic_static.argtypes = [vp, vp, vp, i, i, i, d, d, i, vp]
        L.demag_static_scratch_bytes.argtypes = []
        L.demag_static_scratch_bytes.restype = ctypes.c_size_t
        L.demag_plan_dims.argtypes = [vp, vp, vp, vp, vp]
        L.demag_llg_create.argtypes = [ctypes.POINTER(vp), vp, d, d, d]
        L.demag_llg_set_field.argtypes = [vp, d, d, d]
        L.demag_llg_step.argtypes = [vp, vp, d, i, vp]
        L.demag_llg_mean.argtypes = [vp, vp, vp, vp]
        L.demag_llg_counts.argtypes = [vp, vp, vp, vp]
        L.demag_llg_reset.argtypes = [vp]
        L.demag_llg_destroy.argtypes = [vp]
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
        L.demag_set_pbc_images.argtypes = [vp, i]
        L.demag_extrapolate.argtypes = [vp, i, vp, vp, d, vp, i, vp]
        L.demag_shard_range.argtypes = [i, i, i, i, vp, vp]
        L.demag_plan_create_sharded.argtypes = [ctypes.POINTER(vp), i, i, i, d, d, d, u, i, i, i]
        L.demag_shard_info.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.demag_shard_buffers.argtypes = [vp, vp, vp, vp, vp]
        L.demag_shard_ipc_export.argtypes = [vp, vp]
        L.demag_shard_ipc_connect.argtypes = [vp, vp]
        L.demag_shard_set_peers.argtypes = [vp, vp, vp]
        L.demag_apply_sharded.argtypes = [vp, i, vp, vp, vp]
        for name in EXPORTS:
            if name not in ("demag_workspace_bytes", "demag_launches_per_apply", "demag_last_error", "demag_static_scratch_bytes"):
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


def demag_extrapolate(plan, H_hist, t_hist, t, H_out, accumulate=False, stream=None):
    n = len(H_hist)
    ptrs = (ctypes.c_void_p * n)(*[h.data_ptr() for h in H_hist])
    ts = (ctypes.c_double * n)(*[float(v) for v in t_hist])
    _check(lib().demag_extrapolate(plan, n, ctypes.addressof(ptrs), ctypes.addressof(ts), float(t), H_out.data_ptr(),
                                   int(bool(accumulate)), _stream(stream)))


def demag_energy(plan, M, H, E, stream=None):
    _check(lib().demag_energy(plan, M.data_ptr(), H.data_ptr(), E.data_ptr(), _stream(stream)))


def demag_apply_atomistic(plan, S, Hs, c, mu_s, a, accumulate=False, stream=None):
    _check(lib().demag_apply_atomistic(plan, S.data_ptr(), Hs.data_ptr(), int(c[0]), int(c[1]), int(c[2]),
                                       float(mu_s), float(a), int(bool(accumulate)), _stream(stream)))


def demag_apply_atomistic_static(plan, S, Hs, c, mu_s, a, accumulate=False, stream=None):
    """demag_apply_atomistic with the macrocell arrays in the library's fixed static device array: allocates nothing."""
    _check(lib().demag_apply_atomistic_static(plan, S.data_ptr(), Hs.data_ptr(), int(c[0]), int(c[1]), int(c[2]),
                                              float(mu_s), float(a), int(bool(accumulate)), _stream(stream)))


def demag_static_scratch_bytes() -> int:
    return int(lib().demag_static_scratch_bytes())


def demag_atomistic_reserve(plan):
    _check(lib().demag_atomistic_reserve(plan))


def demag_get_kernel_real(plan, n) -> np.ndarray:
    nx, ny, nz = n
    out = np.empty((6, nz, ny, nx), dtype=np.float64)
    _check(lib().demag_get_kernel_real(plan, out.ctypes.data))
    return out


def demag_workspace_bytes(plan) -> int:
    return int(lib().demag_workspace_bytes(plan))


def demag_set_slab(plan, kx_per_slab: int):
    _check(lib().demag_set_slab(plan, int(kx_per_slab)))


def demag_set_pbc_images(plan, images: int):
    _check(lib().demag_set_pbc_images(plan, int(images)))


def demag_launches_per_apply(plan) -> int:
    return int(lib().demag_launches_per_apply(plan))


def demag_path(plan) -> int:
    return int(lib().demag_path(plan))


def demag_plan_destroy(plan):
    _check(lib().demag_plan_destroy(plan))


# ---- several GPUs (include/demag.h "Several GPUs"): one rank per process ------------------------------------
IPC_BYTES = 128


def demag_shard_range(n, world, rank, align=1):
    """-> (begin, count) of `rank`'s units; host arithmetic only."""
    b, c = ctypes.c_int(), ctypes.c_int()
    _check(lib().demag_shard_range(int(n), int(world), int(rank), int(align), ctypes.addressof(b), ctypes.addressof(c)))
    return b.value, c.value


def demag_plan_create_sharded(nx, ny, nz, hx, hy, hz, pbc_flags, precision, rank, world) -> int:
    h = ctypes.c_void_p()
    _check(lib().demag_plan_create_sharded(ctypes.byref(h), int(nx), int(ny), int(nz), float(hx), float(hy), float(hz),
                                           int(pbc_flags), int(precision), int(rank), int(world)))
    return h.value


def demag_shard_info(plan) -> dict:
    v = [ctypes.c_int() for _ in range(6)]
    _check(lib().demag_shard_info(plan, *[ctypes.addressof(x) for x in v]))
    return dict(zip(("rank", "world", "y0", "ny_loc", "q0", "nq_loc"), (x.value for x in v)))


def demag_shard_buffers(plan):
    """-> (w1in_ptr, w1in_bytes, w1out_ptr, w1out_bytes)"""
    a, b = ctypes.c_void_p(), ctypes.c_void_p()
    na, nb = ctypes.c_size_t(), ctypes.c_size_t()
    _check(lib().demag_shard_buffers(plan, ctypes.addressof(a), ctypes.addressof(na), ctypes.addressof(b), ctypes.addressof(nb)))
    return a.value, na.value, b.value, nb.value


def demag_shard_ipc_export(plan) -> bytes:
    buf = (ctypes.c_ubyte * IPC_BYTES)()
    _check(lib().demag_shard_ipc_export(plan, ctypes.addressof(buf)))
    return bytes(buf)


def demag_shard_ipc_connect(plan, all_handles: bytes):
    buf = (ctypes.c_ubyte * len(all_handles)).from_buffer_copy(all_handles)
    _check(lib().demag_shard_ipc_connect(plan, ctypes.addressof(buf)))


def demag_shard_set_peers(plan, w1in_of_rank, w1out_of_rank):
    n = len(w1in_of_rank)
    a = (ctypes.c_void_p * n)(*w1in_of_rank)
    b = (ctypes.c_void_p * n)(*w1out_of_rank)
    _check(lib().demag_shard_set_peers(plan, ctypes.addressof(a), ctypes.addressof(b)))


def demag_apply_sharded(plan, phase, M_loc=None, H_loc=None, stream=None):
    _check(lib().demag_apply_sharded(plan, int(phase), M_loc.data_ptr() if M_loc is not None else None,
                                     H_loc.data_ptr() if H_loc is not None else None, _stream(stream)))


def gather_handles(handle_bytes: bytes, group=None) -> bytes:
    """All-gather of the ranks' IPC exports over torch.distributed (any backend), rank-major."""
    import torch.distributed as dist
    out = [None] * dist.get_world_size(group)
    dist.all_gather_object(out, handle_bytes, group=group)
    return b"".join(out)


class ShardedPlan:
    """One rank of the partitioned convolution.  `apply` runs the three phases with a barrier over the process
    group between them; the barrier is an all-reduce of one element enqueued on the current stream (NCCL), so
    the host never waits."""

    def __init__(self, n, h, precision=DEMAG_FP32, rank=None, world=None, group=None, connect=True):
        import torch
        import torch.distributed as dist
        self.group = group
        if rank is None:
            rank, world = dist.get_rank(group), dist.get_world_size(group)
        self.n, self.h, self.precision, self.rank, self.world = tuple(n), tuple(h), precision, rank, world
        self.handle = demag_plan_create_sharded(*n, *h, 0, precision, rank, world)
        self.info = demag_shard_info(self.handle)
        self._flag = None
        if connect:
            if world == 1:
                a, _, b, _ = demag_shard_buffers(self.handle)
                demag_shard_set_peers(self.handle, [a], [b])
            else:
                demag_shard_ipc_connect(self.handle, gather_handles(demag_shard_ipc_export(self.handle), group))
                self._flag = torch.zeros(1, device="cuda")

    def local_shape(self):
        nx, ny, nz = self.n
        return (3, nz, self.info["ny_loc"], nx)

    def set_kernel(self, N6_host=None):
        demag_set_kernel(self.handle, N6_host)
        return self

    def barrier(self, stream=None):
        """Order this rank's peer stores before the peers' reads: an all-reduce of one element enqueued on the SAME
        stream the phases run on (torch enqueues collectives on its current stream)."""
        if self.world > 1:
            import torch
            import torch.distributed as dist
            if stream is None:
                dist.all_reduce(self._flag, group=self.group)
            else:
                with torch.cuda.stream(stream):
                    dist.all_reduce(self._flag, group=self.group)

    def apply(self, M_loc, H_loc, stream=None):
        demag_apply_sharded(self.handle, 0, M_loc, None, stream)
        self.barrier(stream)
        demag_apply_sharded(self.handle, 1, None, None, stream)
        self.barrier(stream)
        demag_apply_sharded(self.handle, 2, None, H_loc, stream)

    def energy(self, M_loc, H_loc, E, stream=None):
        """E <- the whole mesh's energy on every rank (partial sums all-reduced)."""
        demag_energy(self.handle, M_loc, H_loc, E, stream)
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(E, group=self.group)

    def workspace_bytes(self):
        return demag_workspace_bytes(self.handle)

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

    def extrapolate(self, H_hist, t_hist, t, H_out, accumulate=False, stream=None):
        demag_extrapolate(self.handle, H_hist, t_hist, t, H_out, accumulate, stream)

    def reserve_atomistic(self):
        """Allocate the macrocell arrays apply_atomistic works on (once per plan; apply_atomistic never allocates)."""
        demag_atomistic_reserve(self.handle)
        return self

    def apply_atomistic(self, S, Hs, c, mu_s, a, accumulate=False, stream=None):
        demag_apply_atomistic(self.handle, S, Hs, c, mu_s, a, accumulate, stream)

    def apply_atomistic_static(self, S, Hs, c, mu_s, a, accumulate=False, stream=None):
        demag_apply_atomistic_static(self.handle, S, Hs, c, mu_s, a, accumulate, stream)

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

    def set_pbc_images(self, images):
        demag_set_pbc_images(self.handle, images)

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


GAMMA_LLG = 2.212761569e5      # mu0 |gamma_e| in m / (A s)  (include/demag.h "Minimal time integrator")


def demag_plan_dims(plan) -> dict:
    nx, ny, nz, pr = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(lib().demag_plan_dims(plan, ctypes.byref(nx), ctypes.byref(ny), ctypes.byref(nz), ctypes.byref(pr)))
    return {"n": (nx.value, ny.value, nz.value), "precision": pr.value}


def demag_llg_create(plan, Ms, alpha, gamma=GAMMA_LLG) -> int:
    h = ctypes.c_void_p()
    _check(lib().demag_llg_create(ctypes.byref(h), plan, float(Ms), float(alpha), float(gamma)))
    return h.value


def demag_llg_set_field(llg, H):
    _check(lib().demag_llg_set_field(llg, float(H[0]), float(H[1]), float(H[2])))


def demag_llg_step(llg, M, dt, extrapolate=False, stream=None):
    _check(lib().demag_llg_step(llg, M.data_ptr(), float(dt), int(bool(extrapolate)), _stream(stream)))


def demag_llg_mean(llg, M, out3, stream=None):
    _check(lib().demag_llg_mean(llg, M.data_ptr(), out3.data_ptr(), _stream(stream)))


def demag_llg_counts(llg) -> dict:
    a, b, t = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_double()
    _check(lib().demag_llg_counts(llg, ctypes.byref(a), ctypes.byref(b), ctypes.byref(t)))
    return {"convolutions": a.value, "extrapolations": b.value, "time": t.value}


def demag_llg_reset(llg):
    _check(lib().demag_llg_reset(llg))


def demag_llg_destroy(llg):
    lib().demag_llg_destroy(llg)


class LLG:
    """RK4 integrator of the LLG equation on top of a Plan (include/demag.h demag_llg_*).  Argument
    marshalling only: every stage runs in the library's kernels."""

    def __init__(self, plan: "Plan", Ms, alpha, gamma=GAMMA_LLG):
        self.handle = demag_llg_create(plan.handle, Ms, alpha, gamma)
        self.plan = plan

    def set_field(self, H):
        demag_llg_set_field(self.handle, H)
        return self

    def step(self, M, dt, extrapolate=False, stream=None):
        demag_llg_step(self.handle, M, dt, extrapolate, stream)

    def mean(self, M, out3, stream=None):
        demag_llg_mean(self.handle, M, out3, stream)

    def counts(self):
        return demag_llg_counts(self.handle)

    def reset(self):
        demag_llg_reset(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            demag_llg_destroy(self.handle)
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
