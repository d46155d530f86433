"""ctypes front end of the CPU oracle (oracle/spgpe_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It imports
nothing from paper_2010_15069_b200 and shares no code with the CUDA path.

All arithmetic lives in the C file; this module only marshals numpy arrays
(psi: complex128 [ny, nx, 2]; fields: float64 [ny, nx] or None).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spgpe_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


class OrcParams(ctypes.Structure):
    _fields_ = [
        ("nx", ctypes.c_int), ("ny", ctypes.c_int),
        ("Lx", ctypes.c_double), ("Ly", ctypes.c_double),
        ("g_uu", ctypes.c_double), ("g_dd", ctypes.c_double), ("g_ud", ctypes.c_double),
        ("k_L", ctypes.c_double),
        ("norm_mode", ctypes.c_int), ("naive_max", ctypes.c_int), ("rs_split", ctypes.c_int),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_max_threads.restype = ctypes.c_int
    return _lib


def _dp(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(ctypes.c_void_p)


def _psi_ptr(psi: np.ndarray):
    assert psi.dtype == np.complex128 and psi.flags.c_contiguous
    return psi.ctypes.data_as(ctypes.c_void_p)


def params(nx, ny, Lx, Ly, g_uu=0.0, g_dd=0.0, g_ud=0.0, k_L=0.0, norm_mode=0, naive_max=32,
           rs_split=0) -> OrcParams:
    return OrcParams(int(nx), int(ny), float(Lx), float(Ly), float(g_uu), float(g_dd), float(g_ud),
                     float(k_L), int(norm_mode), int(naive_max), int(rs_split))


def params_of(w, naive_max=32, rs_split=0) -> OrcParams:
    """OrcParams of a workloads.Workload."""
    return params(w.nx, w.ny, w.Lx, w.Ly, w.g_uu, w.g_dd, w.g_ud, w.k_L, w.norm_mode, naive_max, rs_split)


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def kgrid(n: int, L: float) -> np.ndarray:
    k = np.empty(n)
    lib().orc_kgrid(int(n), ctypes.c_double(L), _dp(k))
    return k


def xgrid(n: int, L: float) -> np.ndarray:
    x = np.empty(n)
    lib().orc_xgrid(int(n), ctypes.c_double(L), _dp(x))
    return x


def dft_naive(a: np.ndarray, sign: int) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    out = np.empty_like(a)
    lib().orc_dft_naive(_psi_ptr(a), _psi_ptr(out), int(a.size), int(sign))
    return out


def fft_radix2(a: np.ndarray, sign: int) -> np.ndarray:
    out = np.array(a, dtype=np.complex128, order="C", copy=True)
    lib().orc_fft_radix2(_psi_ptr(out), int(out.size), int(sign))
    return out


def fft2(psi: np.ndarray, p: OrcParams, sign: int) -> np.ndarray:
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    assert out.shape == (p.ny, p.nx, 2)
    lib().orc_fft2(_psi_ptr(out), ctypes.byref(p), int(sign))
    return out


def su2(a: float, bx: float, bz: float, tau: float, imag: int) -> np.ndarray:
    U = np.empty(4, dtype=np.complex128)
    lib().orc_su2(ctypes.c_double(a), ctypes.c_double(bx), ctypes.c_double(bz), ctypes.c_double(tau),
                  int(imag), _psi_ptr(U))
    return U.reshape(2, 2)


def half(psi, V, Om, de, p: OrcParams, tau: float, imag: int) -> np.ndarray:
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    lib().orc_half(_psi_ptr(out), _dp(V), _dp(Om), _dp(de), ctypes.byref(p), ctypes.c_double(tau), int(imag))
    return out


def kinetic_tables(p: OrcParams):
    a, b, c = np.empty(p.nx), np.empty(p.nx), np.empty(p.ny)
    lib().orc_kinetic_tables(ctypes.byref(p), _dp(a), _dp(b), _dp(c))
    return a, b, c


def kinetic(psi, p: OrcParams, dt: float, imag: int) -> np.ndarray:
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    lib().orc_kinetic(_psi_ptr(out), ctypes.byref(p), ctypes.c_double(dt), int(imag))
    return out


def norm(psi, p: OrcParams) -> np.ndarray:
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    out = np.empty(2)
    lib().orc_norm(_psi_ptr(psi), ctypes.byref(p), _dp(out))
    return out


def step(psi, V, Om, de, p: OrcParams, n: int, dt: float, imag: int,
         targets: Optional[Sequence[float]] = None) -> np.ndarray:
    """n Strang steps; returns a new array.  targets default to the norms of the input."""
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    t = np.array(norm(out, p) if targets is None else targets, dtype=np.float64)
    lib().orc_step(_psi_ptr(out), _dp(V), _dp(Om), _dp(de), ctypes.byref(p), int(n), ctypes.c_double(dt),
                   int(imag), _dp(t))
    return out


def energy(psi, V, Om, de, p: OrcParams) -> np.ndarray:
    """[total, kinetic, potential+Zeeman, interaction, Raman]"""
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    out = np.empty(5)
    lib().orc_energy(_psi_ptr(psi), _dp(V), _dp(Om), _dp(de), ctypes.byref(p), _dp(out))
    return out


def half_nested(psi, V, Om, de, p: OrcParams, tau: float, imag: int) -> np.ndarray:
    """D(tau/2) X(tau) D(tau/2) whatever p.rs_split says."""
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    lib().orc_half_nested(_psi_ptr(out), _dp(V), _dp(Om), _dp(de), ctypes.byref(p), ctypes.c_double(tau), int(imag))
    return out


def anneal_noise(psi, p: OrcParams, seed: int, event: int, amp: float) -> np.ndarray:
    """psi + the Gaussian noise of annealing event `event` (counter-based generator of the C file)."""
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    lib().orc_anneal_noise(_psi_ptr(out), ctypes.byref(p), ctypes.c_ulonglong(seed & 0xFFFFFFFFFFFFFFFF),
                           ctypes.c_longlong(event), ctypes.c_double(amp))
    return out


def step_anneal(psi, V, Om, de, p: OrcParams, n: int, dt: float, every: int, amp: float, seed: int,
                first_step: int = 0, targets: Optional[Sequence[float]] = None) -> np.ndarray:
    """n imaginary-time steps; noise event j/every enters step j when j > 0 and j % every == 0."""
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    t = np.array(norm(out, p) if targets is None else targets, dtype=np.float64)
    lib().orc_step_anneal(_psi_ptr(out), _dp(V), _dp(Om), _dp(de), ctypes.byref(p), int(n), ctypes.c_double(dt),
                          _dp(t), ctypes.c_longlong(first_step), int(every), ctypes.c_double(amp),
                          ctypes.c_ulonglong(seed & 0xFFFFFFFFFFFFFFFF))
    return out


def observables(psi, p: OrcParams) -> np.ndarray:
    """[N_up, N_dn, I_uu, I_dd, I_ud, s] (Eq. 14)."""
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    out = np.empty(6)
    lib().orc_observables(_psi_ptr(psi), ctypes.byref(p), _dp(out))
    return out


def kspace_observables(hat, p: OrcParams) -> np.ndarray:
    """[M_up, M_dn, T_up, T_dn, P_up, P_dn] of a forward-transformed order parameter."""
    hat = np.ascontiguousarray(hat, dtype=np.complex128)
    out = np.empty(6)
    lib().orc_kspace_observables(_psi_ptr(hat), ctypes.byref(p), _dp(out))
    return out


def step_observe(psi, V, Om, de, p: OrcParams, n: int, dt: float, imag: int,
                 targets: Optional[Sequence[float]] = None):
    """(psi after n steps, real-space observables of it, k-space observables in the middle of the last step)."""
    out = np.array(psi, dtype=np.complex128, order="C", copy=True)
    t = np.array(norm(out, p) if targets is None else targets, dtype=np.float64)
    o_r, o_k = np.empty(6), np.empty(6)
    lib().orc_step_observe(_psi_ptr(out), _dp(V), _dp(Om), _dp(de), ctypes.byref(p), int(n), ctypes.c_double(dt),
                           int(imag), _dp(t), _dp(o_r), _dp(o_k))
    return out, o_r, o_k
