"""Test-side helpers: numpy restatements of the packed layouts of include/tmw.h and expected values derived from
the oracle. Nothing here is used by the product; nothing here comes from the CUDA path.
"""
from __future__ import annotations

import numpy as np

import oracle
from paper_2201_09004_b200 import synth


def parity_sites(L: int, T: int, par: int) -> np.ndarray:
    """Lexicographic indices (x fastest) of the sites with (x+y+z+t) % 2 == par, ascending: entry cb is the site
    with checkerboard index cb = lex // 2."""
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    mask = ((x + y + z + t) % 2 == par).ravel()
    lex = np.nonzero(mask)[0]
    assert np.array_equal(lex // 2, np.arange(lex.size))
    return lex


def _planes(a: np.ndarray, dtype) -> np.ndarray:
    """(Vh, nreal) reals -> (NP, Vh, N) planes of 16-byte vectors, zero padded."""
    n = 4 if dtype == np.float32 else 2
    vh, nreal = a.shape
    npl = (nreal + n - 1) // n
    buf = np.zeros((vh, npl * n), dtype=dtype)
    buf[:, :nreal] = a.astype(dtype)
    return np.ascontiguousarray(buf.reshape(vh, npl, n).transpose(1, 0, 2))


def pack_spinor(psi: np.ndarray, par: int, dtype) -> np.ndarray:
    """canonical (T,L,L,L,4,3) complex128 -> packed parity spinor (NP, Vh, N)."""
    T, L = psi.shape[0], psi.shape[1]
    flat = np.ascontiguousarray(psi).reshape(-1, 12).view(np.float64).reshape(-1, 24)
    return _planes(flat[parity_sites(L, T, par)], dtype)


def unpack_spinor(packed: np.ndarray, par: int, L: int, T: int, out: np.ndarray | None = None) -> np.ndarray:
    """packed (NP, Vh, N) -> writes the sites of parity par of a canonical complex128 spinor."""
    if out is None:
        out = np.zeros((T, L, L, L, 4, 3), dtype=np.complex128)
    npl, vh, n = packed.shape
    reals = packed.transpose(1, 0, 2).reshape(vh, npl * n)[:, :24].astype(np.float64)
    flat = out.reshape(-1, 12).view(np.float64).reshape(-1, 24)
    flat[parity_sites(L, T, par)] = reals
    return out


def pack_gauge(U: np.ndarray, par: int, ng: int, dtype) -> np.ndarray:
    """canonical (4,T,L,L,L,3,3) -> (4, NP, Vh, N): the first ng reals (rows 0,1 [,2]) of each link on parity par."""
    T, L = U.shape[1], U.shape[2]
    sites = parity_sites(L, T, par)
    out = []
    for mu in range(4):
        flat = np.ascontiguousarray(U[mu]).reshape(-1, 9).view(np.float64).reshape(-1, 18)
        out.append(_planes(flat[sites][:, :ng], dtype))
    return np.stack(out)


def site_diagonal_blocks(gauge: np.ndarray, c_sw: float, m_re: float) -> np.ndarray:
    """The Hermitian part C(x) = (c_sw/2) sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x) - (4 + Re m) of the site-diagonal
    term, from the oracle's F and sigma, as (V, 2, 6, 6): chirality blocks, index 3*(spin mod 2) + colour."""
    T, L = gauge.shape[1], gauge.shape[2]
    V = L ** 3 * T
    F = oracle.field_strength(gauge)  # (V, 6, 3, 3)
    full = np.zeros((V, 4, 3, 4, 3), dtype=np.complex128)
    plane = 0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            sig = oracle.sigma(mu, nu)
            full += 0.5 * c_sw * np.einsum("st,vab->vsatb", sig, F[:, plane])
            plane += 1
    full = full.reshape(V, 12, 12)
    full += -(4.0 + m_re) * np.eye(12)
    assert np.max(np.abs(full[:, :6, 6:])) < 1e-14 and np.max(np.abs(full[:, 6:, :6])) < 1e-14
    return np.stack([full[:, :6, :6], full[:, 6:, 6:]], axis=1)


def pack_hermitian(blocks: np.ndarray) -> np.ndarray:
    """(..., 6, 6) Hermitian -> (..., 36): 6 real diagonal, then strictly-lower entries row-major as re, im."""
    out = np.empty(blocks.shape[:-2] + (36,), dtype=np.float64)
    for i in range(6):
        out[..., i] = blocks[..., i, i].real
    k = 6
    for i in range(1, 6):
        for j in range(i):
            out[..., k] = blocks[..., i, j].real
            out[..., k + 1] = blocks[..., i, j].imag
            k += 2
    return out


def per_site_rel_err(got: np.ndarray, ref: np.ndarray):
    """max over sites of |got(x) - ref(x)|_2 / |ref(x)|_2 over the 12 components (sites with ref = 0 must be
    exactly 0 in got and are excluded), and the global relative L2 error."""
    g = got.reshape(-1, 12)
    r = ref.reshape(-1, 12)
    rn = np.linalg.norm(r, axis=1)
    dn = np.linalg.norm(g - r, axis=1)
    zero = rn == 0
    assert np.all(dn[zero] == 0), "sites where the reference vanishes must be exactly zero"
    site = float(np.max(dn[~zero] / rn[~zero])) if np.any(~zero) else 0.0
    glob = float(np.linalg.norm(g - r) / max(np.linalg.norm(r), 1e-300))
    return site, glob


def exact_eigenvector_case(L=4, T=8):
    """A system on which BiCGStab is exact at its first half step, IN FLOATING POINT: unit links except U_t = -1 on the last
    time slice (which undoes the antiperiodic wrap of C6, so a constant spinor is an eigenvector), m = -2, a constant source
    with entries in {0, +-1/2, +-1, +-2}. Every hop term is then +-psi or +-i psi times 1/2, summed to 4 psi; the site term is
    -(4 + m) psi = -2 psi; so D b = 2 b, alpha = 1/2, s = r - alpha v = 0, <t,t> = 0, all without a rounding error.
    Returns (U, b); the solution is b / 2."""
    U = synth.unit_gauge(L, T).copy()
    U[3, T - 1] *= -1.0
    u = np.array([[1, -2, 0.5], [0.5j, 1 + 1j, -1], [2j, 0, -0.5 + 1j], [-1, 0.5, 2 - 0.5j]], dtype=np.complex128)
    b = np.ascontiguousarray(np.broadcast_to(u, (T, L, L, L, 4, 3))).copy()
    return U, b
