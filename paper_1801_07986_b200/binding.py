"""Thin Python binding of libpn.so (include/pn.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C-ABI; PyTorch supplies device
memory (fp64 CUDA tensors of shape (N, 3)) and the stream.  There is no CPU fallback: loading
fails loudly if the shared library is missing, and pn_create fails without a CUDA device.
Function names mirror the C entry points.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

PKG = Path(__file__).resolve().parent
LIB_PATH = PKG / "libpn.so"

PN_OK, PN_EINVAL, PN_ECUDA, PN_ESTATE, PN_ENOMEM = 0, -1, -2, -3, -4
PN_OPT_PAIR_PRECISION, PN_OPT_USE_GRAPH, PN_OPT_TIME_PAIR, PN_OPT_J_SPLIT, PN_OPT_PAIR_KERNEL, PN_OPT_EQUAL_MASS, PN_OPT_CROSS_TERMS = 1, 2, 3, 4, 5, 6, 7
PN_CROSS_STAR, PN_CROSS_BH = 1, 2
PN_FP64, PN_FP32_PAIR = 0, 1
PN_PAIR_AUTO, PN_PAIR_TILED, PN_PAIR_SYMMETRIC = 0, 1, 2

# every symbol include/pn.h declares (tests check that the library exports all of them)
EXPORTS = (
    "pn_create", "pn_destroy", "pn_set_stream", "pn_set_option", "pn_set_state", "pn_get_state",
    "pn_set_state_host", "pn_get_state_host", "pn_accel", "pn_accel_host", "pn_step", "pn_energy", "pn_momentum",
    "pn_get_launch_count", "pn_get_pair_time", "pn_get_pair_config", "pn_last_error",
    "pn_version", "pn_bh_accel_noalloc", "pn_get_epilogue_time",
)
PN_NOALLOC_MAX_STARS = 1 << 20

_lib = None


class PNError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libpn error {code}: {msg}")
        self.code = code


def load_library() -> ctypes.CDLL:
    """dlopen libpn.so and declare the signatures.  Raises if the extension has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1801_07986_b200.build` "
            "(nvcc, sm_100a).  This package has no CPU fallback."
        )
    lib = ctypes.CDLL(str(LIB_PATH))
    vp, i64, dbl, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
    lib.pn_create.argtypes = [ctypes.POINTER(vp), i64, vp, dbl, dbl, dbl]
    lib.pn_destroy.argtypes = [vp]
    lib.pn_set_stream.argtypes = [vp, vp]
    lib.pn_set_option.argtypes = [vp, ci, ci]
    for name in ("pn_set_state", "pn_get_state", "pn_set_state_host", "pn_get_state_host"):
        getattr(lib, name).argtypes = [vp, vp, vp]
    lib.pn_accel.argtypes = [vp, vp, vp, vp]
    lib.pn_accel_host.argtypes = [vp, vp, vp, vp]
    lib.pn_step.argtypes = [vp, dbl, i64]
    lib.pn_energy.argtypes = [vp, ctypes.POINTER(dbl)]
    lib.pn_momentum.argtypes = [vp, ctypes.POINTER(dbl)]
    lib.pn_get_launch_count.argtypes = [vp, ctypes.POINTER(i64)]
    lib.pn_get_pair_time.argtypes = [vp, ctypes.POINTER(dbl), ctypes.POINTER(i64), ci]
    lib.pn_get_epilogue_time.argtypes = [vp, ctypes.POINTER(dbl), ctypes.POINTER(i64), ci]
    lib.pn_get_pair_config.argtypes = [vp, ctypes.POINTER(ctypes.c_int32)]
    lib.pn_last_error.argtypes = [vp]
    lib.pn_last_error.restype = ctypes.c_char_p
    lib.pn_version.argtypes = []
    lib.pn_bh_accel_noalloc.argtypes = [i64, vp, vp, vp, dbl, dbl, vp, vp, ctypes.c_char_p, ctypes.c_size_t]
    lib.pn_version.restype = ctypes.c_char_p
    for name in EXPORTS:
        if name not in ("pn_last_error", "pn_version"):
            getattr(lib, name).restype = ci
    _lib = lib
    return lib


def pn_version() -> str:
    return load_library().pn_version().decode()


def _check(lib, ctx, rc: int):
    if rc != PN_OK:
        raise PNError(rc, lib.pn_last_error(ctx).decode())


def _dev_ptr(t, n: int, name: str) -> int:
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or tuple(t.shape) != (n, 3) \
            or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous CUDA float64 tensor of shape ({n}, 3)")
    return t.data_ptr()


def _host_ptr(a, n: int, name: str) -> int:
    """numpy array or CPU torch tensor (e.g. pinned), float64, C-contiguous, shape (n, 3)."""
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or a.shape != (n, 3) or not a.flags.c_contiguous:
            raise TypeError(f"{name} must be a C-contiguous float64 array of shape ({n}, 3)")
        return a.ctypes.data
    import torch

    if isinstance(a, torch.Tensor) and not a.is_cuda and a.dtype == torch.float64 and tuple(a.shape) == (n, 3) \
            and a.is_contiguous():
        return a.data_ptr()
    raise TypeError(f"{name} must be a host float64 array/tensor of shape ({n}, 3)")


def pn_bh_accel_noalloc(masses, pos, vel, G: float, c: float, a1, stream=None):
    """a_1 (Eqs. 2.1 + 2.2) through the library's one entry point that allocates no device memory.

    It exists for callers that cannot call cudaMalloc -- their own pool owns the GPU's memory, they run under a memory
    quota, or they sit in a loop that cannot take cudaMalloc's device-wide stall -- so it needs no PN context and the
    CALLER supplies every tensor, the output included: masses (N,), pos and vel (N, 3), a1 (3,), all contiguous CUDA
    float64.  At most PN_NOALLOC_MAX_STARS = 2**20 stars (the library's fixed scratch array); PNError(PN_EINVAL) beyond.
    Asynchronous on `stream` (default: torch's current stream).  The first call on a device does a one-time set-up and
    should come before any stream capture; calls that overlap on the GPU share the scratch array and race (pn.h).
    Marshalling only: this function creates no tensor."""
    import torch

    lib = load_library()
    n = int(masses.shape[0]) if hasattr(masses, "shape") and len(masses.shape) == 1 else -1
    for t, shape, name in ((masses, (n,), "masses"), (a1, (3,), "a1")):
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or tuple(t.shape) != shape \
                or not t.is_contiguous():
            raise TypeError(f"{name} must be a contiguous CUDA float64 tensor of shape {shape}")
    if stream is None:
        stream = torch.cuda.current_stream()
    handle = getattr(stream, "cuda_stream", stream)
    err = ctypes.create_string_buffer(512)
    rc = lib.pn_bh_accel_noalloc(n, masses.data_ptr(), _dev_ptr(pos, n, "pos"), _dev_ptr(vel, n, "vel"), float(G), float(c),
                                 a1.data_ptr(), ctypes.c_void_p(int(handle)), err, len(err))
    if rc != PN_OK:
        raise PNError(rc, err.value.decode())
    return a1


class PN:
    """One pn_ctx.  Body 0 is the massive object: masses[0] = M."""

    def __init__(self, masses, G: float, c: float, softening: float, stream=None):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p(None)
        m = np.ascontiguousarray(masses, dtype=np.float64)
        if m.ndim != 1:
            raise TypeError("masses must be one-dimensional")
        self.N = int(m.shape[0])
        rc = self._lib.pn_create(ctypes.byref(self._ctx), self.N, m.ctypes.data, float(G), float(c), float(softening))
        if rc != PN_OK:
            self._ctx = ctypes.c_void_p(None)
            raise PNError(rc, self._lib.pn_last_error(None).decode())
        self.pn_set_stream(stream)

    # ---- C entry points, same names -------------------------------------------------------------------
    def pn_set_stream(self, stream=None):
        """stream: torch.cuda.Stream, raw cudaStream_t int, or None for torch's current stream."""
        if stream is None:
            import torch

            stream = torch.cuda.current_stream()
        handle = getattr(stream, "cuda_stream", stream)
        _check(self._lib, self._ctx, self._lib.pn_set_stream(self._ctx, ctypes.c_void_p(int(handle))))

    def pn_set_option(self, key: int, value: int):
        _check(self._lib, self._ctx, self._lib.pn_set_option(self._ctx, int(key), int(value)))

    def pn_set_state(self, pos, vel):
        _check(self._lib, self._ctx, self._lib.pn_set_state(self._ctx, _dev_ptr(pos, self.N, "pos"), _dev_ptr(vel, self.N, "vel")))

    def pn_get_state(self, pos=None, vel=None):
        import torch

        if pos is None:
            pos = torch.empty((self.N, 3), dtype=torch.float64, device="cuda")
        if vel is None:
            vel = torch.empty((self.N, 3), dtype=torch.float64, device="cuda")
        _check(self._lib, self._ctx, self._lib.pn_get_state(self._ctx, _dev_ptr(pos, self.N, "pos"), _dev_ptr(vel, self.N, "vel")))
        return pos, vel

    def pn_set_state_host(self, pos, vel):
        _check(self._lib, self._ctx, self._lib.pn_set_state_host(self._ctx, _host_ptr(pos, self.N, "pos"), _host_ptr(vel, self.N, "vel")))

    def pn_get_state_host(self, pos=None, vel=None):
        if pos is None:
            pos = np.empty((self.N, 3), dtype=np.float64)
        if vel is None:
            vel = np.empty((self.N, 3), dtype=np.float64)
        _check(self._lib, self._ctx, self._lib.pn_get_state_host(self._ctx, _host_ptr(pos, self.N, "pos"), _host_ptr(vel, self.N, "vel")))
        return pos, vel

    def pn_accel(self, pos, vel, acc=None):
        import torch

        if acc is None:
            acc = torch.empty((self.N, 3), dtype=torch.float64, device=pos.device)
        _check(self._lib, self._ctx,
               self._lib.pn_accel(self._ctx, _dev_ptr(pos, self.N, "pos"), _dev_ptr(vel, self.N, "vel"), _dev_ptr(acc, self.N, "acc")))
        return acc

    def pn_accel_host(self, pos, vel, acc=None):
        if acc is None:
            acc = np.empty((self.N, 3), dtype=np.float64)
        _check(self._lib, self._ctx,
               self._lib.pn_accel_host(self._ctx, _host_ptr(pos, self.N, "pos"), _host_ptr(vel, self.N, "vel"), _host_ptr(acc, self.N, "acc")))
        return acc

    def pn_step(self, dt: float, nsteps: int = 1):
        _check(self._lib, self._ctx, self._lib.pn_step(self._ctx, float(dt), int(nsteps)))

    def pn_energy(self) -> float:
        e = ctypes.c_double(0.0)
        _check(self._lib, self._ctx, self._lib.pn_energy(self._ctx, ctypes.byref(e)))
        return e.value

    def pn_momentum(self) -> np.ndarray:
        out = (ctypes.c_double * 3)()
        _check(self._lib, self._ctx, self._lib.pn_momentum(self._ctx, out))
        return np.array(list(out), dtype=np.float64)

    def pn_get_launch_count(self) -> int:
        n = ctypes.c_int64(0)
        _check(self._lib, self._ctx, self._lib.pn_get_launch_count(self._ctx, ctypes.byref(n)))
        return n.value

    def pn_get_pair_time(self, reset: bool = True):
        ms, n = ctypes.c_double(0.0), ctypes.c_int64(0)
        _check(self._lib, self._ctx, self._lib.pn_get_pair_time(self._ctx, ctypes.byref(ms), ctypes.byref(n), int(reset)))
        return ms.value, n.value

    def pn_get_epilogue_time(self, reset: bool = True):
        ms, n = ctypes.c_double(0.0), ctypes.c_int64(0)
        _check(self._lib, self._ctx, self._lib.pn_get_epilogue_time(self._ctx, ctypes.byref(ms), ctypes.byref(n), int(reset)))
        return ms.value, n.value

    def pn_get_pair_config(self) -> dict:
        cfg = (ctypes.c_int32 * 8)()
        _check(self._lib, self._ctx, self._lib.pn_get_pair_config(self._ctx, cfg))
        keys = ("threads", "i_per_thread", "j_tile", "j_splits", "grid_blocks", "padded_stars", "fp64_instr_per_pair", "variant")
        return dict(zip(keys, list(cfg)))

    def pn_destroy(self):
        if self._ctx:
            self._lib.pn_destroy(self._ctx)
            self._ctx = ctypes.c_void_p(None)

    # ---- conveniences ---------------------------------------------------------------------------------
    close = pn_destroy

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.pn_destroy()

    def __del__(self):
        try:
            self.pn_destroy()
        except Exception:
            pass
