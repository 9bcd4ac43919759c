"""Seeded synthetic inputs (harness side): random SU(3) gauge fields and source spinors.

This module holds none of the method's arithmetic. It produces numpy arrays in the canonical user-facing
layouts of ``include/tmw.h`` that are handed, unchanged, to BOTH the CPU oracle and the CUDA library, so that
bit-identical inputs never depend on either implementation.

Canonical layouts (fp64, x fastest):
  gauge  [mu=0..3 (x,y,z,t)][t][z][y][x][row][col]   complex128
  spinor [t][z][y][x][spin 0..3][colour 0..2]         complex128
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth.c")
_LIB = os.path.join(_HERE, "libsynth.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile synth.c with gcc (plain C + OpenMP) into libsynth.so next to it."""
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
        i64, u64, dbl, ptr = ctypes.c_int64, ctypes.c_uint64, ctypes.c_double, ctypes.c_void_p
        lib.synth_su3.argtypes = [i64, dbl, u64, u64, i64, ptr]
        lib.synth_gauge.argtypes = [ctypes.c_int, ctypes.c_int, dbl, u64, ptr]
        lib.synth_z2.argtypes = [i64, u64, ptr]
        lib.synth_gauss.argtypes = [i64, u64, ptr]
        for f in (lib.synth_su3, lib.synth_gauge, lib.synth_z2, lib.synth_gauss):
            f.restype = None
        _lib = lib
    return _lib


def volume(L: int, T: int) -> int:
    return L * L * L * T


def gauge_field(L: int, T: int, eps: float, seed: int = 1) -> np.ndarray:
    """Random SU(3) links U = exp(i eps H), re-unitarised; shape (4, T, L, L, L, 3, 3) complex128."""
    out = np.empty((4, T, L, L, L, 3, 3), dtype=np.complex128)
    _load().synth_gauge(L, T, float(eps), seed, out.ctypes.data)
    return out


def su3_matrices(n: int, eps: float, seed: int, stream: int = 7) -> np.ndarray:
    """n random SU(3) matrices (e.g. a gauge transformation g(x)); shape (n, 3, 3)."""
    out = np.empty((n, 3, 3), dtype=np.complex128)
    _load().synth_su3(n, float(eps), seed, stream, 0, out.ctypes.data)
    return out


def unit_gauge(L: int, T: int) -> np.ndarray:
    out = np.zeros((4, T, L, L, L, 3, 3), dtype=np.complex128)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
    return out


def point_source(L: int, T: int, spin: int = 0, colour: int = 0, site=(0, 0, 0, 0)) -> np.ndarray:
    """b(x)_{s,c} = delta_{x,site} delta_{s,spin} delta_{c,colour}; site = (x,y,z,t)."""
    b = np.zeros((T, L, L, L, 4, 3), dtype=np.complex128)
    x, y, z, t = site
    b[t, z, y, x, spin, colour] = 1.0
    return b


def z2_source(L: int, T: int, seed: int = 2) -> np.ndarray:
    """Each of the 12V components is +-1 + 0i with equal probability."""
    out = np.empty((T, L, L, L, 4, 3), dtype=np.complex128)
    _load().synth_z2(out.size, seed, out.ctypes.data)
    return out


def gaussian_spinor(L: int, T: int, seed: int = 3) -> np.ndarray:
    out = np.empty((T, L, L, L, 4, 3), dtype=np.complex128)
    _load().synth_gauss(out.size, seed, out.ctypes.data)
    return out


# The five BASELINE.json configs (shapes and parameters of the paper's Table 1 ensembles).
CONFIGS = [
    dict(name="cfg0_4x8", L=4, T=8, m=(0.1, 0.0), c_sw=0.0, eps=0.3, source="point"),
    dict(name="cfg1_24x64_tm", L=24, T=64, m=(-0.0695, 0.01), c_sw=0.0, eps=0.4, source="z2"),
    dict(name="cfg2_24x64_clover", L=24, T=64, m=(-0.0695, 0.0), c_sw=1.0509, eps=0.4, source="point"),
    dict(name="cfg3_32x96_clover", L=32, T=96, m=(-0.0514, 0.0), c_sw=1.0424, eps=0.35, source="point12"),
    dict(name="cfg4_48x144_clover", L=48, T=144, m=(-0.0398, 0.0), c_sw=1.0349, eps=0.3, source="point"),
]
