"""Thin ctypes binding of libtmw.so (include/tmw.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels. There is no CPU fallback: loading fails loudly when
libtmw.so is missing, and every call raises TmwError on a non-zero return code.

torch is used here only to obtain device pointers / the current stream from torch tensors; numpy arrays are
passed as HOST pointers (the context must then have been created with location=HOST).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtmw.so")

OK, EINVAL, ENOMEM, ECUDA, ESINGULAR, ENOCONV, EBREAKDOWN = 0, -1, -2, -3, -4, -5, -6
DEVICE, HOST = 0, 1
MIXED, DOUBLE = 0, 1
BICGSTAB, GCR = 0, 1
TWIST_GAMMA5, MASS_SCALAR = 0, 1
D, DDAG, G5D = 0, 1, 2
FULL, EVEN, ODD = 0, 1, 2
F32, F64 = 0, 1
DEBUG_FORCE_PIVOT, DEBUG_NO_CHUNK, DEBUG_FORCE_DEFECT = 1, 2, 4
STATIC_SCRATCH_BYTES = 8 << 20  # TMW_STATIC_SCRATCH_BYTES
# kernel kinds of tmw_kernel_counts / tmw_time_kernel (include/tmw.h TMW_K_*)
KINDS = ["hop32", "k1_32", "k2_32", "k2_32_dots", "hop64", "k1_64", "k2_64", "xpay64", "ainvxpay64", "update_s", "update_xrp",
         "acc_y", "resid_convert", "convert", "dot_norm64", "sub_norm", "diag64", "pack_both", "unpack_both", "other",
         "memset_bytes", "copy_bytes", "hop32_loadonly", "staged", "ffma_probe", "ffma2_probe"]
FFMA_PROBE_FMAS_PER_THREAD = 16 * 16384

EXPORTS = ["tmw_create", "tmw_apply", "tmw_apply_schur", "tmw_apply_schur_static", "tmw_solve", "tmw_apply_multi", "tmw_apply_schur_multi",
           "tmw_solve_multi", "tmw_cheb_apply", "tmw_spinor_bytes", "tmw_pack", "tmw_unpack",
           "tmw_get_clover", "tmw_set_location", "tmw_set_debug", "tmw_launch_count", "tmw_kernel_counts",
           "tmw_time_kernel", "tmw_destroy", "tmw_last_error"]


class tmw_complex(ctypes.Structure):
    _fields_ = [("re", ctypes.c_double), ("im", ctypes.c_double)]


class tmw_options(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_size_t), ("location", ctypes.c_int), ("precision", ctypes.c_int), ("reconstruct", ctypes.c_int),
                ("mass_reading", ctypes.c_int), ("max_iter", ctypes.c_int), ("delta", ctypes.c_double),
                ("stream", ctypes.c_void_p), ("solver", ctypes.c_int), ("nkrylov", ctypes.c_int),
                ("verbose", ctypes.c_int), ("columns_per_thread", ctypes.c_int),
                ("tile", ctypes.c_int * 4), ("debug", ctypes.c_int), ("domains_z", ctypes.c_int), ("domains_t", ctypes.c_int),
                ("stage", ctypes.c_int), ("stage_tile", ctypes.c_int * 3), ("zchunk", ctypes.c_int), ("prefetch", ctypes.c_int)]


def make_options(**fields) -> tmw_options:
    """tmw_options with struct_size set (what TMW_OPTIONS_INIT does in C) and the given members; the rest stay 0 = default."""
    opt = tmw_options()
    opt.struct_size = ctypes.sizeof(tmw_options)
    for k, v in fields.items():
        if k not in {f[0] for f in tmw_options._fields_} or k == "struct_size":
            raise TypeError(f"tmw_options has no member {k!r}")
        setattr(opt, k, v)
    return opt


class tmw_solve_info(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("reliable_updates", ctypes.c_int), ("restarts", ctypes.c_int),
                ("iter_resid", ctypes.c_double), ("true_resid", ctypes.c_double), ("device_ms", ctypes.c_double)]


class TmwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"tmw error {code}: {msg}")
        self.code = code


_lib = None


def load():
    """dlopen libtmw.so and declare the prototypes of include/tmw.h. Raises if the library was not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2201_09004_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    P, I, DBL, LL = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong
    lib.tmw_create.argtypes = [ctypes.POINTER(P), I, I, P, tmw_complex, DBL, ctypes.POINTER(tmw_options)]
    lib.tmw_create.restype = I
    lib.tmw_apply.argtypes = [P, I, I, I, P, P]
    lib.tmw_apply.restype = I
    lib.tmw_apply_schur.argtypes = [P, I, I, P, P]
    lib.tmw_apply_schur.restype = I
    lib.tmw_apply_schur_static.argtypes = [P, I, I, P, P]
    lib.tmw_apply_schur_static.restype = I
    lib.tmw_solve.argtypes = [P, P, P, DBL, ctypes.POINTER(tmw_solve_info)]
    lib.tmw_solve.restype = I
    lib.tmw_apply_multi.argtypes = [P, I, I, I, I, P, P]
    lib.tmw_apply_multi.restype = I
    lib.tmw_apply_schur_multi.argtypes = [P, I, I, I, P, P]
    lib.tmw_apply_schur_multi.restype = I
    lib.tmw_solve_multi.argtypes = [P, I, P, P, DBL, ctypes.POINTER(tmw_solve_info)]
    lib.tmw_solve_multi.restype = I
    lib.tmw_cheb_apply.argtypes = [P, I, ctypes.POINTER(DBL), DBL, DBL, P, P]
    lib.tmw_cheb_apply.restype = I
    lib.tmw_spinor_bytes.argtypes = [P, I]
    lib.tmw_spinor_bytes.restype = LL
    lib.tmw_pack.argtypes = [P, I, I, P, P]
    lib.tmw_pack.restype = I
    lib.tmw_unpack.argtypes = [P, I, I, P, P]
    lib.tmw_unpack.restype = I
    lib.tmw_get_clover.argtypes = [P, I, I, P]
    lib.tmw_get_clover.restype = I
    lib.tmw_set_location.argtypes = [P, I]
    lib.tmw_set_location.restype = I
    lib.tmw_set_debug.argtypes = [P, I]
    lib.tmw_set_debug.restype = I
    lib.tmw_launch_count.argtypes = [P]
    lib.tmw_launch_count.restype = LL
    lib.tmw_kernel_counts.argtypes = [P, ctypes.POINTER(LL), I]
    lib.tmw_kernel_counts.restype = I
    lib.tmw_time_kernel.argtypes = [P, I, I, ctypes.POINTER(DBL)]
    lib.tmw_time_kernel.restype = I
    lib.tmw_destroy.argtypes = [P]
    lib.tmw_destroy.restype = None
    lib.tmw_last_error.argtypes = [P]
    lib.tmw_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _ptr(a):
    """address of a torch tensor (device or host) or a numpy array"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    if isinstance(a, int):
        return a
    assert a.is_contiguous()
    return a.data_ptr()


class Context:
    """Owns a tmw_ctx. Methods mirror the C entry points: create (constructor), apply, apply_schur, solve, pack,
    unpack, get_clover, destroy."""

    def __init__(self, L: int, T: int, gauge, m: complex, c_sw: float = 0.0, *, location: int = DEVICE,
                 precision: int = MIXED, reconstruct: int = 12, mass_reading: int = TWIST_GAMMA5, max_iter: int = 0,
                 delta: float = 0.0, stream: int | None = None, solver: int = BICGSTAB, nkrylov: int = 0,
                 verbose: int = 0, columns_per_thread: int = 0, tile=(0, 0, 0, 0), debug: int = 0, domains_z: int = 0, domains_t: int = 0,
                 stage: int = 0, stage_tile=(0, 0, 0), zchunk: int = 0, prefetch: int = 0):
        lib = load()
        self._lib = lib
        self.L, self.T = L, T
        self.V = L * L * L * T
        self.location = location
        opt = make_options(location=location, precision=precision, reconstruct=reconstruct, mass_reading=mass_reading,
                           max_iter=max_iter, delta=delta, stream=stream, solver=solver, nkrylov=nkrylov, verbose=verbose,
                           columns_per_thread=columns_per_thread, tile=(ctypes.c_int * 4)(*tile), debug=debug,
                           domains_z=domains_z, domains_t=domains_t, stage=stage,
                           stage_tile=(ctypes.c_int * 3)(*stage_tile), zchunk=zchunk, prefetch=prefetch)
        h = ctypes.c_void_p()
        rc = lib.tmw_create(ctypes.byref(h), L, T, _ptr(gauge), tmw_complex(float(np.real(m)), float(np.imag(m))),
                            float(c_sw), ctypes.byref(opt))
        if rc != OK:
            raise TmwError(rc, (lib.tmw_last_error(None) or b"").decode())
        self._h = h

    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise TmwError(rc, (self._lib.tmw_last_error(self._h) or b"").decode())
        return rc

    def apply(self, op: int, parity: int, prec: int, src, dst):
        self._check(self._lib.tmw_apply(self._h, op, parity, prec, _ptr(src), _ptr(dst)))

    def apply_schur(self, op: int, prec: int, src, dst):
        self._check(self._lib.tmw_apply_schur(self._h, op, prec, _ptr(src), _ptr(dst)))

    def apply_schur_static(self, op: int, prec: int, src, dst):
        """tmw_apply_schur_static: apply_schur for callers that must not allocate device memory (a pool allocator owns
        the card, a memory quota, a loop that cannot take cudaMalloc's device-wide stall). The intermediate lives in the
        8 MiB array built into libtmw.so (STATIC_SCRATCH_BYTES); larger parity spinors raise TmwError(EINVAL). All
        calls on a device share that array, so keep them on one stream; see include/tmw.h."""
        self._check(self._lib.tmw_apply_schur_static(self._h, op, prec, _ptr(src), _ptr(dst)))

    def solve(self, b, x, tol: float, allow_noconv: bool = False) -> dict:
        info = tmw_solve_info()
        rc = self._check(self._lib.tmw_solve(self._h, _ptr(b), _ptr(x), float(tol), ctypes.byref(info)),
                         allow=(ENOCONV,) if allow_noconv else ())
        return dict(status=rc, iters=info.iters, reliable_updates=info.reliable_updates, restarts=info.restarts,
                    iter_resid=info.iter_resid, true_resid=info.true_resid, device_ms=info.device_ms)

    def apply_multi(self, op: int, parity: int, prec: int, nrhs: int, src, dst):
        self._check(self._lib.tmw_apply_multi(self._h, op, parity, prec, nrhs, _ptr(src), _ptr(dst)))

    def apply_schur_multi(self, op: int, prec: int, nrhs: int, src, dst):
        self._check(self._lib.tmw_apply_schur_multi(self._h, op, prec, nrhs, _ptr(src), _ptr(dst)))

    def solve_multi(self, nrhs: int, b, x, tol: float, allow_noconv: bool = False) -> list:
        infos = (tmw_solve_info * nrhs)()
        rc = self._check(self._lib.tmw_solve_multi(self._h, nrhs, _ptr(b), _ptr(x), float(tol), infos),
                         allow=(ENOCONV,) if allow_noconv else ())
        return [dict(status=rc, iters=i.iters, reliable_updates=i.reliable_updates, restarts=i.restarts,
                     iter_resid=i.iter_resid, true_resid=i.true_resid, device_ms=i.device_ms) for i in infos]

    def cheb_apply(self, coef, scale: float, shift: float, src, dst):
        c = (ctypes.c_double * len(coef))(*[float(v) for v in coef])
        self._check(self._lib.tmw_cheb_apply(self._h, len(coef), c, float(scale), float(shift), _ptr(src), _ptr(dst)))

    def spinor_bytes(self, prec: int) -> int:
        return int(self._lib.tmw_spinor_bytes(self._h, prec))

    def pack(self, prec: int, parity: int, canonical, packed):
        self._check(self._lib.tmw_pack(self._h, prec, parity, _ptr(canonical), _ptr(packed)))

    def unpack(self, prec: int, parity: int, packed, canonical):
        self._check(self._lib.tmw_unpack(self._h, prec, parity, _ptr(packed), _ptr(canonical)))

    def get_clover(self, parity: int, inverse: int, dst):
        self._check(self._lib.tmw_get_clover(self._h, parity, inverse, _ptr(dst)))

    def set_location(self, location: int):
        self._check(self._lib.tmw_set_location(self._h, location))
        self.location = location

    def set_debug(self, flags: int):
        self._check(self._lib.tmw_set_debug(self._h, flags))

    def launch_count(self) -> int:
        return int(self._lib.tmw_launch_count(self._h))

    def kernel_counts(self) -> dict:
        buf = (ctypes.c_longlong * len(KINDS))()
        n = self._lib.tmw_kernel_counts(self._h, buf, len(KINDS))
        if n != len(KINDS):
            raise TmwError(n, "tmw_kernel_counts: kind table out of date")
        return {k: int(v) for k, v in zip(KINDS, buf)}

    def time_kernel(self, kind: str, reps: int = 20) -> float:
        ms = ctypes.c_double(0.0)
        self._check(self._lib.tmw_time_kernel(self._h, KINDS.index(kind), reps, ctypes.byref(ms)))
        return ms.value

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.tmw_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()
