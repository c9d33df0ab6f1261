"""ctypes loader for the ORACLE (test infrastructure, not the product).

`oracle/lgf_oracle.cpp` is the plain serial-semantics C++ implementation of the method
(SURVEY.md §8(c)); this file only compiles it with g++ and marshals numpy arrays.
Only tests/, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs
may import this package; nothing under `paper_1208_1186_b200/` does.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lgf_oracle.cpp")
_SO = os.path.join(_HERE, "liblgf_oracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2 -fopenmp).  Returns the path of the shared library."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _SO + ".tmp", _SRC]
        subprocess.run(cmd, check=True)
        os.replace(_SO + ".tmp", _SO)
    return _SO


_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_threads.restype = ctypes.c_int
        _lib.orc_fix.restype = ctypes.c_int64
        _lib.orc_fix.argtypes = [_ip, _dp, ctypes.c_double, ctypes.c_double, ctypes.c_int64, _dp, _dp, _dp, _dp]
        _lib.orc_iterate.argtypes = [_ip, _dp, ctypes.c_int64, ctypes.c_double, _dp, _dp]
        _lib.orc_build_g.argtypes = [_ip, _dp, ctypes.c_double, _dp]
        _lib.orc_two_row_roundtrip.argtypes = [ctypes.c_int64, _dp, _dp]
        _lib.orc_wilson_lines.argtypes = [_ip, _dp, _dp]
        _lib.orc_singlet_correlator.argtypes = [_ip, _dp, _dp]
    return _lib


def _d(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _L(L: Sequence[int]):
    return (ctypes.c_int32 * 4)(*[int(v) for v in L])


def _vol(L) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def _f64(a) -> np.ndarray:
    """torch tensor / ndarray (real view [..., 2] or complex) -> contiguous float64 ndarray copy."""
    if hasattr(a, "detach"):
        a = a.detach().cpu().numpy()
    a = np.asarray(a)
    if np.iscomplexobj(a):
        a = np.ascontiguousarray(a.astype(np.complex128)).view(np.float64)
    return np.array(a, dtype=np.float64, order="C", copy=True)


def threads() -> int:
    return int(lib().orc_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def dft1d(x: np.ndarray, sign: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    lib().orc_dft1d(len(x), _d(x.view(np.float64)), _d(out.view(np.float64)), int(sign))
    return out


def fft1d(x: np.ndarray, sign: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    lib().orc_fft1d(len(x), _d(x.view(np.float64)), _d(out.view(np.float64)), int(sign))
    return out


def transform4d(L, f: np.ndarray, sign: int, direct: bool = False) -> np.ndarray:
    """f: complex [V] (x fastest).  sign=-1 forward unnormalised; +1 inverse with 1/V."""
    out = np.array(f, dtype=np.complex128, order="C", copy=True).reshape(-1)
    assert out.size == _vol(L)
    lib().orc_transform4d(_L(L), _d(out.view(np.float64)), int(sign), int(direct))
    return out


def psq(L) -> Tuple[np.ndarray, float]:
    p2 = np.empty(_vol(L), dtype=np.float64)
    pmax = ctypes.c_double()
    lib().orc_psq(_L(L), _d(p2), ctypes.byref(pmax))
    return p2, pmax.value


def measure(L, U) -> Tuple[np.ndarray, float, float]:
    """-> (Delta complex [V,3,3], theta, F)."""
    U = _f64(U)
    V = _vol(L)
    assert U.size == V * 72
    D = np.empty(V * 18, dtype=np.float64)
    th, F = ctypes.c_double(), ctypes.c_double()
    lib().orc_measure(_L(L), _d(U), _d(D), ctypes.byref(th), ctypes.byref(F))
    return D.view(np.complex128).reshape(V, 3, 3), th.value, F.value


def fourier_accelerate(L, Delta, direct: bool = False) -> np.ndarray:
    D = _f64(Delta)
    V = _vol(L)
    assert D.size == V * 18
    out = np.empty(V * 18, dtype=np.float64)
    lib().orc_fourier_accelerate(_L(L), _d(D), _d(out), int(direct))
    return out.view(np.complex128).reshape(V, 3, 3)


def build_g(L, Dtilde, alpha: float) -> np.ndarray:
    D = _f64(Dtilde)
    V = _vol(L)
    out = np.empty(V * 18, dtype=np.float64)
    lib().orc_build_g(_L(L), _d(D), float(alpha), _d(out))
    return out.view(np.complex128).reshape(V, 3, 3)


def reunitarise(m) -> np.ndarray:
    a = _f64(m)
    out = np.empty(18, dtype=np.float64)
    lib().orc_reunitarise(_d(a), _d(out))
    return out.view(np.complex128).reshape(3, 3)


def update_links(L, U, g) -> np.ndarray:
    U, g = _f64(U), _f64(g)
    V = _vol(L)
    out = np.empty(V * 72, dtype=np.float64)
    lib().orc_update_links(_L(L), _d(U), _d(g), _d(out))
    return out.view(np.complex128).reshape(V, 4, 3, 3)


def two_row_roundtrip(U) -> np.ndarray:
    U = _f64(U)
    out = np.empty_like(U)
    lib().orc_two_row_roundtrip(U.size // 18, _d(U), _d(out))
    return out.view(np.complex128).reshape(-1, 4, 3, 3)


def iterate(L, U, n: int, alpha: float):
    """-> (links complex [V,4,3,3] after n updates, theta_hist[n+1], F_hist[n+1])."""
    U = _f64(U)
    th = np.empty(n + 1, dtype=np.float64)
    Fh = np.empty(n + 1, dtype=np.float64)
    lib().orc_iterate(_L(L), _d(U), int(n), float(alpha), _d(th), _d(Fh))
    return U.view(np.complex128).reshape(_vol(L), 4, 3, 3), th, Fh


def fix(L, U, alpha: float, theta_tol: float, max_iter: int):
    """-> (links, iterations, theta, F, theta_hist[:iterations+1], F_hist[:iterations+1])."""
    U = _f64(U)
    th = np.empty(max_iter + 1, dtype=np.float64)
    Fh = np.empty(max_iter + 1, dtype=np.float64)
    t, F = ctypes.c_double(), ctypes.c_double()
    n = lib().orc_fix(_L(L), _d(U), float(alpha), float(theta_tol), int(max_iter),
                      ctypes.byref(t), ctypes.byref(F), _d(th), _d(Fh))
    return (U.view(np.complex128).reshape(_vol(L), 4, 3, 3), int(n), t.value, F.value,
            th[:n + 1].copy(), Fh[:n + 1].copy())


def wilson_lines(L, U) -> np.ndarray:
    """Temporal Wilson lines W(x) = prod_t U_t(x, t) -> complex [Vs, 3, 3], Vs = Lx Ly Lz."""
    U = _f64(U)
    Vs = _vol(L) // int(L[3])
    out = np.empty(Vs * 18, dtype=np.float64)
    lib().orc_wilson_lines(_L(L), _d(U), _d(out))
    return out.view(np.complex128).reshape(Vs, 3, 3)


def singlet_correlator(L, U) -> np.ndarray:
    """C(r) = (1/(3 Vs)) sum_x Tr[W(x + r) W(x)^+] -> complex [Vs] (x fastest), by the direct double sum (eq. (1))."""
    U = _f64(U)
    Vs = _vol(L) // int(L[3])
    out = np.empty(Vs * 2, dtype=np.float64)
    lib().orc_singlet_correlator(_L(L), _d(U), _d(out))
    return out.view(np.complex128)
