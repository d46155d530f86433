"""paper_2010_15069_b200 -- thin Python binding of libspgpe (include/spgpe.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch supplies
device memory and the stream, nothing else.  There is no CPU fallback: importing works without a GPU (so
that the build and the symbol table can be checked), but creating a solver raises unless libspgpe is built
and an sm_100 device is present.

Functions carry the names of the C ABI (spgpe_create, spgpe_set_potential, ..., spgpe_step, spgpe_norm,
spgpe_energy); device arrays are torch CUDA tensors, host arrays numpy arrays, both in the layout of
include/spgpe.h (psi: complex [ny, nx, 2]; fields: real [ny, nx]).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from . import _build

SPGPE_C128, SPGPE_C64 = 0, 1
SPGPE_NORM_PER_COMPONENT, SPGPE_NORM_TOTAL = 0, 1
SPGPE_RS_EXPONENTIAL, SPGPE_RS_NESTED = 0, 1

# every symbol include/spgpe.h declares (tests check the library exports exactly these)
ABI_SYMBOLS = (
    "spgpe_create", "spgpe_destroy",
    "spgpe_set_potential", "spgpe_set_raman", "spgpe_set_zeeman",
    "spgpe_set_potential_host", "spgpe_set_raman_host", "spgpe_set_zeeman_host",
    "spgpe_set_psi", "spgpe_get_psi", "spgpe_set_psi_host", "spgpe_get_psi_host", "spgpe_set_norm_targets",
    "spgpe_step", "spgpe_step_observe", "spgpe_set_real_space_split", "spgpe_set_annealing",
    "spgpe_norm", "spgpe_norm_noalloc", "spgpe_energy", "spgpe_synchronize", "spgpe_launch_count",
    "spgpe_profile", "spgpe_profile_read",
    "spgpe_strerror", "spgpe_last_cuda_error", "spgpe_probe_dfma", "spgpe_probe_ffma", "spgpe_probe_copy",
)


class SpgpeParams(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int), ("g_uu", ctypes.c_double), ("g_dd", ctypes.c_double),
                ("g_ud", ctypes.c_double), ("k_L", ctypes.c_double), ("norm_mode", ctypes.c_int)]


class SpgpeError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(what)
        self.code = code


_lib = None


def build(force: bool = False) -> str:
    """Compile libspgpe.so in-tree (nvcc, sm_100a)."""
    return _build.build(force=force)


def lib() -> ctypes.CDLL:
    """Load libspgpe.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_build.LIB_PATH):
            raise SpgpeError(-100, f"{_build.LIB_PATH} is missing: run paper_2010_15069_b200.build() "
                                   "(libspgpe has no CPU fallback)")
        L = ctypes.CDLL(_build.LIB_PATH)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.spgpe_create.argtypes = [ctypes.POINTER(vp), ci, ci, cd, cd, ctypes.POINTER(SpgpeParams), vp]
        for name in ("spgpe_set_potential", "spgpe_set_raman", "spgpe_set_zeeman", "spgpe_set_potential_host",
                     "spgpe_set_raman_host", "spgpe_set_zeeman_host", "spgpe_set_psi", "spgpe_get_psi",
                     "spgpe_set_psi_host", "spgpe_get_psi_host"):
            getattr(L, name).argtypes = [vp, vp]
        L.spgpe_destroy.argtypes = [vp]
        L.spgpe_synchronize.argtypes = [vp]
        L.spgpe_set_norm_targets.argtypes = [vp, cd, cd]
        L.spgpe_step.argtypes = [vp, ci, cd, ci]
        L.spgpe_step_observe.argtypes = [vp, ci, cd, ci, ctypes.POINTER(cd)]
        L.spgpe_set_real_space_split.argtypes = [vp, ci]
        L.spgpe_set_annealing.argtypes = [vp, ci, cd, ctypes.c_ulonglong]
        L.spgpe_norm.argtypes = [vp, ctypes.POINTER(cd)]
        L.spgpe_norm_noalloc.argtypes = [vp, ci, ci, ci, cd, cd, vp, vp]
        L.spgpe_energy.argtypes = [vp, ctypes.POINTER(cd)]
        L.spgpe_launch_count.argtypes = [vp]
        L.spgpe_launch_count.restype = ctypes.c_longlong
        L.spgpe_profile.argtypes = [vp, ci]
        L.spgpe_profile_read.argtypes = [vp, ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_longlong)]
        L.spgpe_strerror.argtypes = [ci]
        L.spgpe_strerror.restype = ctypes.c_char_p
        L.spgpe_last_cuda_error.restype = ctypes.c_char_p
        L.spgpe_probe_dfma.argtypes = [vp, ctypes.POINTER(cd)]
        L.spgpe_probe_ffma.argtypes = [vp, ctypes.POINTER(cd)]
        L.spgpe_probe_copy.argtypes = [vp, ctypes.c_longlong, ctypes.POINTER(cd)]
        _lib = L
    return _lib


def _check(rc: int) -> None:
    if rc != 0:
        L = lib()
        msg = L.spgpe_strerror(rc).decode()
        if rc == -4:
            msg += ": " + L.spgpe_last_cuda_error().decode()
        raise SpgpeError(rc, f"libspgpe: {msg}")


def _dev_ptr(t, dtype_ok, shape) -> Optional[int]:
    """Device pointer of a contiguous torch CUDA tensor (None passes NULL)."""
    if t is None:
        return None
    if not (hasattr(t, "is_cuda") and t.is_cuda):
        raise TypeError("expected a torch CUDA tensor (use the *_host call for numpy arrays)")
    if t.dtype not in dtype_ok or tuple(t.shape) != tuple(shape) or not t.is_contiguous():
        raise TypeError(f"expected a contiguous tensor of shape {tuple(shape)} and dtype in {dtype_ok}, "
                        f"got {tuple(t.shape)} {t.dtype}")
    return t.data_ptr()


def _host_ptr(a, dtype, shape) -> Optional[int]:
    if a is None:
        return None
    if not isinstance(a, np.ndarray) or a.dtype != dtype or a.shape != tuple(shape) or not a.flags.c_contiguous:
        raise TypeError(f"expected a C-contiguous numpy array of shape {tuple(shape)} and dtype {dtype}")
    return a.ctypes.data


class Handle:
    """Owner of one spgpe_handle; remembers the shapes/dtypes the C side expects."""

    def __init__(self, ptr, nx, ny, dtype):
        self.ptr, self.nx, self.ny, self.dtype = ptr, nx, ny, dtype

    @property
    def _torch_dtypes(self):
        import torch
        return ((torch.complex128,), (torch.float64,)) if self.dtype == SPGPE_C128 else \
               ((torch.complex64,), (torch.float32,))

    @property
    def _np_dtypes(self):
        return (np.complex128, np.float64) if self.dtype == SPGPE_C128 else (np.complex64, np.float32)

    def __del__(self):
        try:
            if self.ptr:
                lib().spgpe_destroy(self.ptr)
                self.ptr = None
        except Exception:
            pass


def spgpe_create(nx: int, ny: int, Lx: float, Ly: float, dtype: int = SPGPE_C128, g_uu: float = 0.0,
                 g_dd: float = 0.0, g_ud: float = 0.0, k_L: float = 0.0,
                 norm_mode: int = SPGPE_NORM_PER_COMPONENT, stream: Optional[int] = None) -> Handle:
    """stream: a cudaStream_t as an integer (e.g. torch.cuda.current_stream().cuda_stream); None = default."""
    p = SpgpeParams(int(dtype), float(g_uu), float(g_dd), float(g_ud), float(k_L), int(norm_mode))
    out = ctypes.c_void_p()
    _check(lib().spgpe_create(ctypes.byref(out), int(nx), int(ny), float(Lx), float(Ly), ctypes.byref(p),
                              ctypes.c_void_p(stream or 0)))
    return Handle(out, int(nx), int(ny), int(dtype))


def spgpe_destroy(h: Handle) -> None:
    if h.ptr:
        _check(lib().spgpe_destroy(h.ptr))
        h.ptr = None


def _set_field(fn_dev, fn_host, h: Handle, a) -> None:
    if a is None or (hasattr(a, "is_cuda") and a.is_cuda):
        _check(getattr(lib(), fn_dev)(h.ptr, _dev_ptr(a, h._torch_dtypes[1], (h.ny, h.nx))))
    else:
        _check(getattr(lib(), fn_host)(h.ptr, _host_ptr(a, h._np_dtypes[1], (h.ny, h.nx))))


def spgpe_set_potential(h: Handle, V) -> None:
    _set_field("spgpe_set_potential", "spgpe_set_potential_host", h, V)


def spgpe_set_raman(h: Handle, Omega) -> None:
    _set_field("spgpe_set_raman", "spgpe_set_raman_host", h, Omega)


def spgpe_set_zeeman(h: Handle, delta) -> None:
    _set_field("spgpe_set_zeeman", "spgpe_set_zeeman_host", h, delta)


spgpe_set_potential_host = spgpe_set_potential
spgpe_set_raman_host = spgpe_set_raman
spgpe_set_zeeman_host = spgpe_set_zeeman


def spgpe_set_psi(h: Handle, psi) -> None:
    _check(lib().spgpe_set_psi(h.ptr, _dev_ptr(psi, h._torch_dtypes[0], (h.ny, h.nx, 2))))


def spgpe_get_psi(h: Handle, out) -> None:
    _check(lib().spgpe_get_psi(h.ptr, _dev_ptr(out, h._torch_dtypes[0], (h.ny, h.nx, 2))))


def spgpe_set_psi_host(h: Handle, psi: np.ndarray) -> None:
    _check(lib().spgpe_set_psi_host(h.ptr, _host_ptr(psi, h._np_dtypes[0], (h.ny, h.nx, 2))))


def spgpe_get_psi_host(h: Handle, out: Optional[np.ndarray] = None) -> np.ndarray:
    if out is None:
        out = np.empty((h.ny, h.nx, 2), dtype=h._np_dtypes[0])
    _check(lib().spgpe_get_psi_host(h.ptr, _host_ptr(out, h._np_dtypes[0], (h.ny, h.nx, 2))))
    return out


def spgpe_set_norm_targets(h: Handle, n_up: float, n_dn: float) -> None:
    _check(lib().spgpe_set_norm_targets(h.ptr, float(n_up), float(n_dn)))


def spgpe_step(h: Handle, n: int, dt: float, imag: int = 0) -> None:
    _check(lib().spgpe_step(h.ptr, int(n), float(dt), int(imag)))


def spgpe_step_observe(h: Handle, n: int, dt: float, imag: int = 0) -> np.ndarray:
    """n steps; [N_up, N_dn, I_uu, I_dd, I_ud, s, M_up, M_dn, T_up, T_dn, P_up, P_dn] (include/spgpe.h)."""
    out = (ctypes.c_double * 12)()
    _check(lib().spgpe_step_observe(h.ptr, int(n), float(dt), int(imag), out))
    return np.array(out[:])


def spgpe_set_real_space_split(h: Handle, mode: int) -> None:
    _check(lib().spgpe_set_real_space_split(h.ptr, int(mode)))


def spgpe_set_annealing(h: Handle, every: int, amp: float, seed: int) -> None:
    _check(lib().spgpe_set_annealing(h.ptr, int(every), float(amp), ctypes.c_ulonglong(seed & 0xFFFFFFFFFFFFFFFF)))


def spgpe_norm(h: Handle) -> np.ndarray:
    out = (ctypes.c_double * 2)()
    _check(lib().spgpe_norm(h.ptr, out))
    return np.array(out[:])


def spgpe_norm_noalloc(psi, Lx: float, Ly: float, out, stream: Optional[int] = None) -> None:
    """N_up, N_dn of the torch CUDA tensor psi (complex [ny, nx, 2]) into the torch CUDA tensor out (2 float64), on
    `stream` (cudaStream_t as an integer; None = default), without a handle and without any allocation; asynchronous.
    Sizes beyond 8192 per axis raise SpgpeError (code -7).  Argument marshalling only (include/spgpe.h)."""
    import torch
    if not (hasattr(psi, "is_cuda") and psi.is_cuda and psi.dim() == 3 and psi.shape[2] == 2 and psi.is_contiguous()):
        raise TypeError("psi: contiguous torch CUDA tensor of shape [ny, nx, 2]")
    if psi.dtype == torch.complex128:
        dt = SPGPE_C128
    elif psi.dtype == torch.complex64:
        dt = SPGPE_C64
    else:
        raise TypeError("psi: complex128 or complex64")
    if not (hasattr(out, "is_cuda") and out.is_cuda and out.dtype == torch.float64 and out.numel() == 2
            and out.is_contiguous() and out.device == psi.device):
        raise TypeError("out: contiguous torch CUDA tensor of 2 float64 on psi's device")
    _check(lib().spgpe_norm_noalloc(psi.data_ptr(), dt, int(psi.shape[1]), int(psi.shape[0]), float(Lx), float(Ly),
                                    out.data_ptr(), ctypes.c_void_p(stream or 0)))


def spgpe_energy(h: Handle) -> np.ndarray:
    """[total, kinetic, potential+Zeeman, interaction, Raman]"""
    out = (ctypes.c_double * 5)()
    _check(lib().spgpe_energy(h.ptr, out))
    return np.array(out[:])


def spgpe_synchronize(h: Handle) -> None:
    _check(lib().spgpe_synchronize(h.ptr))


def spgpe_launch_count(h: Handle) -> int:
    return int(lib().spgpe_launch_count(h.ptr))


def spgpe_profile(h: Handle, enable: bool) -> None:
    _check(lib().spgpe_profile(h.ptr, int(bool(enable))))


def spgpe_profile_read(h: Handle):
    """(ms[2], count[2]): summed CUDA-event durations and launch counts of the row pass and the column pass."""
    ms = (ctypes.c_double * 2)()
    cnt = (ctypes.c_longlong * 2)()
    _check(lib().spgpe_profile_read(h.ptr, ms, cnt))
    return list(ms), list(cnt)


def spgpe_probe_dfma(stream: Optional[int] = None) -> float:
    out = ctypes.c_double()
    _check(lib().spgpe_probe_dfma(ctypes.c_void_p(stream or 0), ctypes.byref(out)))
    return out.value


def spgpe_probe_ffma(stream: Optional[int] = None) -> float:
    out = ctypes.c_double()
    _check(lib().spgpe_probe_ffma(ctypes.c_void_p(stream or 0), ctypes.byref(out)))
    return out.value


def spgpe_probe_copy(nbytes: int, stream: Optional[int] = None) -> float:
    out = ctypes.c_double()
    _check(lib().spgpe_probe_copy(ctypes.c_void_p(stream or 0), int(nbytes), ctypes.byref(out)))
    return out.value


def from_workload(w, stream: Optional[int] = None, dtype: Optional[str] = None) -> Handle:
    """Solver for a workloads.Workload (fields and psi0 uploaded from the host arrays)."""
    dt = SPGPE_C128 if (dtype or w.dtype) == "c128" else SPGPE_C64
    h = spgpe_create(w.nx, w.ny, w.Lx, w.Ly, dt, w.g_uu, w.g_dd, w.g_ud, w.k_L, w.norm_mode, stream)
    cdt, rdt = h._np_dtypes
    for setter, f in ((spgpe_set_potential, w.V), (spgpe_set_raman, w.Omega), (spgpe_set_zeeman, w.delta)):
        setter(h, None if f is None else np.ascontiguousarray(f, dtype=rdt))
    spgpe_set_psi_host(h, np.ascontiguousarray(w.psi0, dtype=cdt))
    return h
