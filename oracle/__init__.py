"""ctypes binding of the fp64 CPU oracle (oracle/tmw_oracle.c). TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2201_09004_b200 and shares no code with the CUDA path.

All arrays are numpy complex128 in the canonical layouts:
  gauge  (4, T, L, L, L, 3, 3)      spinor (T, L, L, L, 4, 3)      F (V, 6, 3, 3)
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tmw_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

TWIST_GAMMA5 = 0
MASS_SCALAR = 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C11 + OpenMP over the site loop)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        ci, dbl, ptr, i64 = ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_int64
        lib.orc_gamma.argtypes = [ci, ptr]
        lib.orc_sigma.argtypes = [ci, ci, ptr]
        lib.orc_field_strength.argtypes = [ci, ci, ptr, ptr]
        lib.orc_apply.argtypes = [ci, ci, ptr, ptr, dbl, dbl, dbl, ci, ci, ci, ptr, ptr]
        lib.orc_apply_sites.argtypes = [ci, ci, ptr, dbl, dbl, dbl, ci, ci, ci, ptr, i64, ptr, ptr]
        lib.orc_bicgstab.argtypes = [ci, ci, ptr, ptr, dbl, dbl, dbl, ci, ci, ci, ptr, ptr, dbl, ci, ptr, ptr]
        lib.orc_bicgstab.restype = ci
        lib.orc_num_threads.restype = ci
        for f in (lib.orc_gamma, lib.orc_sigma, lib.orc_field_strength, lib.orc_apply, lib.orc_apply_sites):
            f.restype = None
        _lib = lib
    return _lib


def _c(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def _dims(gauge: np.ndarray):
    assert gauge.ndim == 7 and gauge.shape[0] == 4 and gauge.shape[5:] == (3, 3), gauge.shape
    T, L = gauge.shape[1], gauge.shape[2]
    assert gauge.shape[2:5] == (L, L, L)
    return L, T


def gamma(mu: int) -> np.ndarray:
    """gamma_mu for mu = 0..3 (x,y,z,t); mu = 4 gives gamma5 = gx gy gz gt."""
    out = np.empty((4, 4), dtype=np.complex128)
    _load().orc_gamma(mu, out.ctypes.data)
    return out


def sigma(mu: int, nu: int) -> np.ndarray:
    out = np.empty((4, 4), dtype=np.complex128)
    _load().orc_sigma(mu, nu, out.ctypes.data)
    return out


def field_strength(gauge: np.ndarray) -> np.ndarray:
    """F_mu_nu(x) for the six planes (xy,xz,xt,yz,yt,zt); shape (V, 6, 3, 3)."""
    L, T = _dims(gauge)
    gauge = _c(gauge)
    out = np.empty((L * L * L * T, 6, 3, 3), dtype=np.complex128)
    _load().orc_field_strength(L, T, gauge.ctypes.data, out.ctypes.data)
    return out


def apply(gauge, psi, m: complex, c_sw: float = 0.0, dagger: bool = False, F=None,
          mass_reading: int = TWIST_GAMMA5, antiperiodic_t: bool = True) -> np.ndarray:
    """out = D psi (or D^dagger psi) on the full lattice."""
    L, T = _dims(gauge)
    gauge, psi = _c(gauge), _c(psi)
    assert psi.shape == (T, L, L, L, 4, 3), psi.shape
    if F is not None:
        F = _c(F)
    out = np.empty_like(psi)
    _load().orc_apply(L, T, gauge.ctypes.data, F.ctypes.data if F is not None else None, float(np.real(m)),
                      float(np.imag(m)), float(c_sw), int(dagger), int(mass_reading), int(antiperiodic_t),
                      psi.ctypes.data, out.ctypes.data)
    return out


def apply_sites(gauge, psi, sites, m: complex, c_sw: float = 0.0, dagger: bool = False,
                mass_reading: int = TWIST_GAMMA5, antiperiodic_t: bool = True) -> np.ndarray:
    """(D psi)(x) at the listed lexicographic site indices only; shape (n, 4, 3)."""
    L, T = _dims(gauge)
    gauge, psi = _c(gauge), _c(psi)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((sites.size, 4, 3), dtype=np.complex128)
    _load().orc_apply_sites(L, T, gauge.ctypes.data, float(np.real(m)), float(np.imag(m)), float(c_sw), int(dagger),
                            int(mass_reading), int(antiperiodic_t), psi.ctypes.data, sites.size, sites.ctypes.data,
                            out.ctypes.data)
    return out


def bicgstab(gauge, b, m: complex, c_sw: float = 0.0, tol: float = 1e-12, max_iter: int = 10000, dagger: bool = False,
             F=None, mass_reading: int = TWIST_GAMMA5, antiperiodic_t: bool = True):
    """Solve D x = b with full-lattice fp64 BiCGStab. Returns (x, info dict)."""
    L, T = _dims(gauge)
    gauge, b = _c(gauge), _c(b)
    if F is None and c_sw != 0.0:
        F = field_strength(gauge)
    if F is not None:
        F = _c(F)
    x = np.empty_like(b)
    iters = ctypes.c_int(0)
    resid = ctypes.c_double(0.0)
    status = _load().orc_bicgstab(L, T, gauge.ctypes.data, F.ctypes.data if F is not None else None,
                                  float(np.real(m)), float(np.imag(m)), float(c_sw), int(dagger), int(mass_reading),
                                  int(antiperiodic_t), b.ctypes.data, x.ctypes.data, float(tol), int(max_iter),
                                  ctypes.byref(iters), ctypes.byref(resid))
    return x, dict(status=status, iters=iters.value, true_resid=resid.value)


def gamma5_apply(gauge, psi, m: complex, c_sw: float = 0.0, F=None) -> np.ndarray:
    """gamma5 D psi (the operator the paper's overlap work is built on; = H_w when m is real):
    the oracle's D followed by the explicit 4x4 gamma5 = gx gy gz gt on the spin index."""
    return np.einsum("st,...tc->...sc", gamma(4), apply(gauge, psi, m, c_sw, F=F))


def cheb_series(gauge, psi, coef, scale: float, shift: float, m: complex, c_sw: float = 0.0, F=None) -> np.ndarray:
    """sum_k coef[k] T_k(X) psi with X = scale * gamma5 D + shift, by the DEFINITION of the Chebyshev polynomials of the
    first kind: T_0 = 1, T_1 = X, T_{k+1} = 2 X T_k - T_{k-1} (each T_k psi formed explicitly and summed). The CUDA path
    evaluates the same series with the Clenshaw recursion; the two agree up to rounding."""
    X = lambda v: scale * gamma5_apply(gauge, v, m, c_sw, F=F) + shift * v
    psi = _c(psi)
    t_prev, out = psi, coef[0] * psi
    if len(coef) > 1:
        t_cur = X(psi)
        out = out + coef[1] * t_cur
        for k in range(2, len(coef)):
            t_prev, t_cur = t_cur, 2.0 * X(t_cur) - t_prev
            out = out + coef[k] * t_cur
    return out


def num_threads() -> int:
    return int(_load().orc_num_threads())
