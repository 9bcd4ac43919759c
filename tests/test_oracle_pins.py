"""Pins of the fp64 CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

The paper (arXiv:2201.09004) prints no operator value, so every pin is a closed form, an invariant, a special case
or brute force (SURVEY.md §8(c) "Pins"). Each test names the mistake it would catch.
"""
import itertools

import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth

TWO_PI = 2.0 * np.pi


# ----------------------------------------------------------------------------------------------------------
# helpers (closed forms written from the definitions, using the golden gamma matrices — not the oracle's)
# ----------------------------------------------------------------------------------------------------------
def coords(L, T):
    """arrays x,y,z,t of shape (T,L,L,L)"""
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    return x, y, z, t


def momentum(L, T, n, antiperiodic=True):
    nx, ny, nz, nt = n
    return np.array([TWO_PI * nx / L, TWO_PI * ny / L, TWO_PI * nz / L,
                     TWO_PI * (nt + (0.5 if antiperiodic else 0.0)) / T])


def plane_wave(L, T, p, u):
    x, y, z, t = coords(L, T)
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return phase[..., None, None] * u[None, None, None, None, :, :]


def rand_spinor(rng, L, T):
    return rng.standard_normal((T, L, L, L, 4, 3)) + 1j * rng.standard_normal((T, L, L, L, 4, 3))


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def dense_matrix(gauge, m, c_sw=0.0, dagger=False, **kw):
    L, T = gauge.shape[2], gauge.shape[1]
    n = 12 * L ** 3 * T
    F = oracle.field_strength(gauge) if c_sw != 0.0 else None
    M = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for j in range(n):
        e[j] = 1.0
        M[:, j] = oracle.apply(gauge, e.reshape(T, L, L, L, 4, 3), m, c_sw, dagger=dagger, F=F, **kw).ravel()
        e[j] = 0.0
    return M


def abelian_flux_gauge(L, T, mu, nu, k):
    """Uniform abelian flux in the (mu,nu) plane, mu<nu, SURVEY.md §8(c) 'Pins/Clover':
    U_mu(x) = exp(-i B x_nu T3), U_nu(x) = exp(+i B L_nu x_mu T3) on x_nu = L_nu - 1, other links 1,
    B = 2 pi k / (L_mu L_nu), T3 = diag(1,-1,0). Every (mu,nu) plaquette is exp(i B T3)."""
    ext = [L, L, L, T]
    B = TWO_PI * k / (ext[mu] * ext[nu])
    U = synth.unit_gauge(L, T)
    c = coords(L, T)
    t3 = np.array([1.0, -1.0, 0.0])
    ph = -B * c[nu]
    for a in range(3):
        U[mu, ..., a, a] = np.exp(1j * ph * t3[a])
    edge = c[nu] == ext[nu] - 1
    ph2 = B * ext[nu] * c[mu]
    for a in range(3):
        U[nu, ..., a, a] = np.where(edge, np.exp(1j * ph2 * t3[a]), 1.0)
    return U, B


PLANES = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]


# ----------------------------------------------------------------------------------------------------------
# gamma algebra and basis
# ----------------------------------------------------------------------------------------------------------
def test_gamma_matrices_match_golden_and_clifford(gammas):
    """Catches: a wrong entry/sign in any gamma matrix; wrong gamma5 ordering."""
    for mu in range(4):
        assert np.array_equal(oracle.gamma(mu), gammas[mu])
        assert np.allclose(gammas[mu], gammas[mu].conj().T)
    for mu in range(4):
        for nu in range(4):
            anti = gammas[mu] @ gammas[nu] + gammas[nu] @ gammas[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu))
    g5 = gammas[0] @ gammas[1] @ gammas[2] @ gammas[3]
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))
    assert np.allclose(oracle.gamma(4), g5)
    for mu, nu in PLANES:
        s = 0.5j * (gammas[mu] @ gammas[nu] - gammas[nu] @ gammas[mu])
        assert np.allclose(oracle.sigma(mu, nu), s)
        assert np.allclose(s[:2, 2:], 0) and np.allclose(s[2:, :2], 0)  # chiral-block diagonal


# ----------------------------------------------------------------------------------------------------------
# (a) free field: closed-form plane-wave eigenvalues (north_star check (a))
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("m", [0.1 + 0.0j, -0.0695 + 0.01j, -0.3 + 0.25j])
def test_free_field_plane_wave_eigenvalues(m):
    """U = 1: eigenvalues -[Re m + sum(1-cos p)] +- i sqrt(sum sin^2 p + (Im m)^2) with antiperiodic p_t
    (SURVEY.md §8(c) C1, C4, C6). Catches: wrong overall sign, missing 1/2, wrong 4+m, missing antiperiodic
    sign, scalar-vs-gamma5 mass reading, wrong neighbour indexing."""
    L, T = 4, 8
    U = synth.unit_gauge(L, T)
    rng = np.random.default_rng(5)
    for n in [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 2, 3, 5), (3, 1, 2, 7)]:
        p = momentum(L, T, n)
        a = m.real + np.sum(1.0 - np.cos(p))
        b = np.sqrt(np.sum(np.sin(p) ** 2) + m.imag ** 2)
        lam_p, lam_m = -a + 1j * b, -a - 1j * b
        u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi = plane_wave(L, T, p, u)
        d1 = oracle.apply(U, psi, m)
        # project on the two eigenspaces: (D - lam_-) psi is an eigenvector with lam_+ and vice versa
        vp = d1 - lam_m * psi
        vm = d1 - lam_p * psi
        assert np.linalg.norm(vp) > 1e-3 and np.linalg.norm(vm) > 1e-3
        assert rel(oracle.apply(U, vp, m), lam_p * vp) < 1e-12
        assert rel(oracle.apply(U, vm, m), lam_m * vm) < 1e-12


def test_free_field_scalar_mass_reading():
    """Literal alternative of C4: -(4+m)*1 with complex m: eigenvalues -[m + sum(1-cos p)] +- i sqrt(sum sin^2 p)."""
    L, T = 4, 4
    U = synth.unit_gauge(L, T)
    m = -0.2 + 0.3j
    rng = np.random.default_rng(6)
    p = momentum(L, T, (1, 3, 2, 1))
    a = m + np.sum(1.0 - np.cos(p))
    b = np.sqrt(np.sum(np.sin(p) ** 2))
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi = plane_wave(L, T, p, u)
    d1 = oracle.apply(U, psi, m, mass_reading=oracle.MASS_SCALAR)
    for lam, other in ((-a + 1j * b, -a - 1j * b), (-a - 1j * b, -a + 1j * b)):
        v = d1 - other * psi
        assert rel(oracle.apply(U, v, m, mass_reading=oracle.MASS_SCALAR), lam * v) < 1e-12


def test_free_field_dense_spectrum_small():
    """Diagonalise the dense matrix on 2^3 x 4 (L = 2: forward and backward neighbours coincide, C19) and compare
    the full multiset of eigenvalues with the closed form (each 6-fold: 3 colours x 2)."""
    L, T = 2, 4
    m = 0.05 + 0.2j
    M = dense_matrix(synth.unit_gauge(L, T), m)
    ev = np.linalg.eigvals(M)
    expect = []
    for n in itertools.product(range(L), range(L), range(L), range(T)):
        p = momentum(L, T, n)
        a = m.real + np.sum(1.0 - np.cos(p))
        b = np.sqrt(np.sum(np.sin(p) ** 2) + m.imag ** 2)
        expect += [-a + 1j * b] * 6 + [-a - 1j * b] * 6
    expect = np.array(expect)
    assert ev.size == expect.size
    key = lambda v: np.lexsort((np.round(v.imag, 6), np.round(v.real, 6)))
    assert np.max(np.abs(ev[key(ev)] - expect[key(expect)])) < 1e-9


def test_constant_abelian_background():
    """U_mu = diag(e^{i th1}, e^{i th2}, e^{-i(th1+th2)}) constant: closed form with p -> p + theta^c per colour, and
    F = 0 so c_sw must not matter. Catches: colour index transposition, U vs U^dagger on the backward hop."""
    L, T = 4, 4
    rng = np.random.default_rng(7)
    th = rng.uniform(-1, 1, size=(4, 2))
    theta = np.concatenate([th, -(th.sum(axis=1, keepdims=True))], axis=1)  # (mu, colour)
    U = synth.unit_gauge(L, T)
    for mu in range(4):
        for c in range(3):
            U[mu, ..., c, c] = np.exp(1j * theta[mu, c])
    m = -0.1 + 0.07j
    for c_sw in (0.0, 1.3):
        for colour in range(3):
            p = momentum(L, T, (1, 2, 0, 3))
            q = p + theta[:, colour]
            a = m.real + np.sum(1.0 - np.cos(q))
            b = np.sqrt(np.sum(np.sin(q) ** 2) + m.imag ** 2)
            u = np.zeros((4, 3), dtype=np.complex128)
            u[:, colour] = rng.standard_normal(4) + 1j * rng.standard_normal(4)
            psi = plane_wave(L, T, p, u)
            d1 = oracle.apply(U, psi, m, c_sw)
            for lam, other in ((-a + 1j * b, -a - 1j * b), (-a - 1j * b, -a + 1j * b)):
                v = d1 - other * psi
                assert np.linalg.norm(v) > 1e-3
                assert rel(oracle.apply(U, v, m, c_sw), lam * v) < 1e-12


# ----------------------------------------------------------------------------------------------------------
# (b) daggered operator
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c_sw", [0.0, 1.0509])
@pytest.mark.parametrize("reading", [oracle.TWIST_GAMMA5, oracle.MASS_SCALAR])
def test_gamma5_hermiticity_and_adjoint(c_sw, reading):
    """D(m)^dag = g5 D(m*) g5 (north_star check (b)) and <y, D x> = <D^dag y, x>. Catches: wrong projector swap or
    wrong conjugation of the twist in D^dag."""
    L, T = 4, 6
    U = synth.gauge_field(L, T, 0.4, seed=11)
    rng = np.random.default_rng(8)
    x, y = rand_spinor(rng, L, T), rand_spinor(rng, L, T)
    m = -0.07 + 0.13j
    g5 = np.array([1, 1, -1, -1])[:, None]
    lhs = oracle.apply(U, x, m, c_sw, dagger=True, mass_reading=reading)
    rhs = g5 * oracle.apply(U, g5 * x, np.conj(m), c_sw, mass_reading=reading)
    assert rel(lhs, rhs) < 1e-13
    d = oracle.apply(U, x, m, c_sw, mass_reading=reading)
    assert abs(vdot(y, d) - vdot(oracle.apply(U, y, m, c_sw, dagger=True, mass_reading=reading), x)) < 1e-10 * abs(vdot(y, d))


def test_dense_conjugate_transpose_2x2x2x2():
    """Brute force on 2^4: the matrix built from dagger=True equals the conjugate transpose of the matrix of D."""
    U = synth.gauge_field(2, 2, 0.4, seed=3)
    m = 0.1 - 0.2j
    M = dense_matrix(U, m, 1.1)
    Md = dense_matrix(U, m, 1.1, dagger=True)
    assert np.max(np.abs(Md - M.conj().T)) < 1e-13


# ----------------------------------------------------------------------------------------------------------
# twisted-mass reading (C4)
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c_sw", [0.0, 1.0349])
def test_twisted_mass_identity(c_sw):
    """|D(m) psi|^2 = |D(Re m) psi|^2 + (Im m)^2 |psi|^2 holds for the gamma5-twist and fails for the scalar reading."""
    L, T = 4, 4
    U = synth.gauge_field(L, T, 0.35, seed=2)
    rng = np.random.default_rng(9)
    psi = rand_spinor(rng, L, T)
    m = -0.0695 + 0.3j
    n2 = lambda v: np.linalg.norm(v.ravel()) ** 2
    lhs = n2(oracle.apply(U, psi, m, c_sw))
    rhs = n2(oracle.apply(U, psi, m.real, c_sw)) + m.imag ** 2 * n2(psi)
    assert abs(lhs - rhs) < 1e-12 * rhs
    lhs_scalar = n2(oracle.apply(U, psi, m, c_sw, mass_reading=oracle.MASS_SCALAR))
    assert abs(lhs_scalar - rhs) > 1e-4 * rhs
    # Im m = 0 reduces both readings to the Wilson operator
    assert rel(oracle.apply(U, psi, m.real, c_sw), oracle.apply(U, psi, m.real, c_sw, mass_reading=oracle.MASS_SCALAR)) == 0.0


# ----------------------------------------------------------------------------------------------------------
# (c) gauge covariance
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c_sw", [0.0, 1.0424])
def test_gauge_covariance(c_sw):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag, psi' = g psi  =>  D[U'] psi' = g D[U] psi (north_star check (c)).
    Catches: wrong link on the backward hop, missing dagger, wrong neighbour, wrong clover leaf."""
    L, T = 4, 6
    V = L ** 3 * T
    U = synth.gauge_field(L, T, 0.4, seed=1)
    g = synth.su3_matrices(V, 0.9, seed=4).reshape(T, L, L, L, 3, 3)
    Up = np.empty_like(U)
    for mu in range(4):
        axis = 3 - mu  # array axes are (t,z,y,x)
        g_fwd = np.roll(g, -1, axis=axis)
        Up[mu] = np.einsum("...ab,...bc,...dc->...ad", g, U[mu], g_fwd.conj())
    rng = np.random.default_rng(10)
    psi = rand_spinor(rng, L, T)
    psip = np.einsum("...ab,...sb->...sa", g, psi)
    m = -0.05 + 0.02j
    lhs = oracle.apply(Up, psip, m, c_sw)
    rhs = np.einsum("...ab,...sb->...sa", g, oracle.apply(U, psi, m, c_sw))
    assert rel(lhs, rhs) < 1e-13


# ----------------------------------------------------------------------------------------------------------
# clover term
# ----------------------------------------------------------------------------------------------------------
def test_field_strength_vanishes_on_unit_and_pure_gauge():
    L, T = 4, 4
    assert np.max(np.abs(oracle.field_strength(synth.unit_gauge(L, T)))) == 0.0
    g = synth.su3_matrices(L ** 3 * T, 1.0, seed=12).reshape(T, L, L, L, 3, 3)
    U = np.empty((4, T, L, L, L, 3, 3), dtype=np.complex128)
    for mu in range(4):
        U[mu] = np.einsum("...ab,...cb->...ac", g, np.roll(g, -1, axis=3 - mu).conj())
    assert np.max(np.abs(oracle.field_strength(U))) < 1e-14


def test_field_strength_hermitian_and_traceful_definition():
    """F is Hermitian; no trace subtraction is applied (C7): tr F = Im tr Q / 4 is generally non-zero."""
    U = synth.gauge_field(4, 4, 0.4, seed=1)
    F = oracle.field_strength(U)
    assert np.max(np.abs(F - np.conj(np.swapaxes(F, -1, -2)))) < 1e-15
    assert np.max(np.abs(np.trace(F, axis1=-2, axis2=-1))) > 1e-3


@pytest.mark.parametrize("plane", range(6))
def test_uniform_abelian_flux(plane, gammas):
    """Uniform abelian flux in plane (mu,nu): F_mu_nu = sin(B) T3 at every site, all other planes zero, and the site term
    of the operator is (c_sw/2) sigma_mu_nu (x) sin(B) T3. Pins leaf orientation, the 1/(8i), the c_sw/2 prefactor and the
    plane ordering/sign of reading C7."""
    L, T = 4, 8
    mu, nu = PLANES[plane]
    U, B = abelian_flux_gauge(L, T, mu, nu, k=1)
    F = oracle.field_strength(U)
    t3 = np.diag([1.0, -1.0, 0.0])
    for pl in range(6):
        expect = np.sin(B) * t3 if pl == plane else np.zeros((3, 3))
        assert np.max(np.abs(F[:, pl] - expect)) < 1e-14
    rng = np.random.default_rng(13)
    psi = rand_spinor(rng, L, T)
    c_sw = 1.7
    diff = oracle.apply(U, psi, 0.1, c_sw) - oracle.apply(U, psi, 0.1, 0.0)
    sig = 0.5j * (gammas[mu] @ gammas[nu] - gammas[nu] @ gammas[mu])
    expect = 0.5 * c_sw * np.sin(B) * np.einsum("st,ab,...tb->...sa", sig, t3, psi)
    assert rel(diff, expect) < 1e-13


def test_clover_sign_is_the_improving_one():
    """Pins the SIGN and prefactor of the clover term of Eq. (3) relative to the hopping term of Eq. (2)
     to what the term is for: "O(a) improvement". The expected values come from the continuum,
    not from reading C7: for a Dirac operator in a uniform abelian field B in the xy-plane,
    (gamma.D)^2 = D^2 + sum_{mu<nu} sigma_mu_nu F_mu_nu, the lowest Landau level has -D^2 = B and sigma_xy F_xy = -B on
    one spin orientation, so gamma.D has exact zero modes. The Wilson term -(1/2) D^2 of Eq. (2) lifts them to B/2 (an
    O(a) artefact); the clover term at c_sw = 1 must cancel exactly that Pauli term, bringing them back to O(B^2). With the
    wrong sign it doubles the lift to B instead; with a wrong prefactor (c_sw/4, c_sw) the cancellation fails too.

    Lattice: 8^3 x 2, fully periodic (antiperiodic_t=False: zero modes need p_t = 0), m = 0, one flux quantum
    B = 2 pi / 64. Colour 2 is neutral under T3 = diag(1,-1,0) and sees a free field (exact zero modes at m = 0): the
    vectors are restricted to colours 0, 1 (abelian links are colour-diagonal, so this sector is invariant). The operator
    commutes with translations in z and t, so the sector of vectors constant in z and t is invariant as well; it holds
    the lowest modes (every other (p_z, p_t) adds (1 - cos p) >= 0), and in it D is a dense 512 x 512 matrix whose
    singular values are computed exactly. Catches: flipped sign of the clover term (or of sigma, or of F) relative to
    the hopping term, wrong prefactor."""
    L, T = 8, 2
    U, B = abelian_flux_gauge(L, T, 0, 1, k=1)
    assert abs(B - TWO_PI / 64) < 1e-15
    F = oracle.field_strength(U)
    n = L * L * 4 * 2

    def sigma_min(c_sw):
        M = np.empty((n, n), dtype=np.complex128)
        j = 0
        for y in range(L):
            for x in range(L):
                for s in range(4):
                    for c in range(2):
                        psi = np.zeros((T, L, L, L, 4, 3), dtype=np.complex128)
                        psi[:, :, y, x, s, c] = 1.0
                        w = oracle.apply(U, psi, 0.0, c_sw, F=F, antiperiodic_t=False)
                        assert np.max(np.abs(w - w[:1, :1])) < 1e-14 and np.max(np.abs(w[..., 2])) == 0.0  # sector is invariant
                        M[:, j] = w[0, 0, :, :, :, :2].ravel()
                        j += 1
        sv = np.sort(np.linalg.svd(M, compute_uv=False))
        # 4 would-be zero modes: 2 colours x (flux quanta |k| = 1 each) x 2 (the lower-chirality copy): well separated from the rest
        assert sv[4] > 3.0 * B
        return sv[:4]

    s0, sp, sm = sigma_min(0.0), sigma_min(+1.0), sigma_min(-1.0)
    assert np.all(np.abs(s0 - B / 2) < 0.05 * B), s0    # Wilson term alone: lifted to B/2          (measured 0.04851 vs 0.04909)
    assert np.all(np.abs(sm - B) < 0.05 * B), sm        # wrong-sign clover term: lift doubled to B  (measured 0.09752 vs 0.09817)
    assert np.all(sp < 0.1 * s0.min()), sp              # c_sw = +1: cancelled to O(B^2)             (measured 5.0e-4)
    assert np.all(sp < B * B), sp


def test_table1_golden_matches_configs():
    """tests/golden/table1_ensembles.txt holds the MILC rows of Table 1 (OCR-garbled cells read as in
    DESIGN.md C9); synth.CONFIGS[1..4] (= BASELINE.json configs[1..4]) must carry exactly these lattice sizes, masses
    and c_sw. Catches: a mistyped ensemble parameter in the workload table every test and bench.py use."""
    import os
    from conftest import GOLDEN
    rows = {}
    with open(os.path.join(GOLDEN, "table1_ensembles.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            tag, L, T, mass, c_sw = line.split()
            rows[tag] = (int(L), int(T), float(mass), float(c_sw))
    assert set(rows) == {"MILC12", "MILC09", "MILC06"}
    cfgs = synth.CONFIGS
    # config 1 = MILC12 without clover and with a twist; config 2 = MILC12 as printed; 3 = MILC09; 4 = MILC06
    for idx, tag in ((2, "MILC12"), (3, "MILC09"), (4, "MILC06")):
        L, T, mass, c_sw = rows[tag]
        c = cfgs[idx]
        assert (c["L"], c["T"]) == (L, T), (idx, tag)
        assert c["m"] == (mass, 0.0) and c["c_sw"] == c_sw, (idx, tag)
    L, T, mass, _ = rows["MILC12"]
    assert (cfgs[1]["L"], cfgs[1]["T"], cfgs[1]["m"][0], cfgs[1]["c_sw"]) == (L, T, mass, 0.0)
    # Table 2 row 1 quotes m_cri + omega = -0.0398 for the 48^3 x 144 ensemble: the same number as Table 1
    assert rows["MILC06"][2] == -0.0398


def test_clover_term_properties_on_random_field():
    """Site term is Hermitian, spin-traceless, chiral-block diagonal; c_sw = 0 reduces to the no-clover operator;
    precomputed F and on-the-fly F agree; apply_sites agrees with the full application."""
    L, T = 4, 4
    U = synth.gauge_field(L, T, 0.4, seed=1)
    F = oracle.field_strength(U)
    rng = np.random.default_rng(14)
    psi = rand_spinor(rng, L, T)
    a = oracle.apply(U, psi, 0.2, 1.05, F=F)
    b = oracle.apply(U, psi, 0.2, 1.05)
    assert rel(a, b) == 0.0
    sites = np.array([0, 1, 17, 100, L ** 3 * T - 1])
    c = oracle.apply_sites(U, psi, sites, 0.2, 1.05)
    assert np.array_equal(c, a.reshape(-1, 4, 3)[sites])
    # site term as a 12x12 matrix at one site
    s = 37
    blk = np.zeros((12, 12), dtype=np.complex128)
    for pl, (mu, nu) in enumerate(PLANES):
        blk += 0.5 * np.kron(oracle.sigma(mu, nu), F[s, pl])
    assert np.allclose(blk, blk.conj().T)
    assert np.allclose(blk[:6, 6:], 0) and np.allclose(blk[6:, :6], 0)
    assert abs(sum(blk[3 * sp + c, 3 * sp + c] for sp in range(4) for c in [0])) < 1e-14  # spin trace at fixed colour


# ----------------------------------------------------------------------------------------------------------
# (d) solver: dense brute force and Fourier-sum propagator
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c_sw,m", [(0.0, 0.1 + 0.0j), (1.0509, -0.0695 + 0.0j), (1.0, -0.044 + 0.05j)])
def test_bicgstab_vs_dense_lu_2x2x2x2(c_sw, m):
    """north_star check (d): dense-matrix brute-force solve on 2^4."""
    U = synth.gauge_field(2, 2, 0.4, seed=1)
    M = dense_matrix(U, m, c_sw)
    rng = np.random.default_rng(15)
    b = rand_spinor(rng, 2, 2)
    x_lu = np.linalg.solve(M, b.ravel())
    x, info = oracle.bicgstab(U, b, m, c_sw, tol=1e-13)
    assert info["status"] == 0 and info["true_resid"] < 1e-12
    assert rel(x.ravel(), x_lu) < 1e-11


def test_bicgstab_vs_dense_lu_4x4x4x4():
    L = T = 4
    U = synth.gauge_field(L, T, 0.4, seed=1)
    m, c_sw = -0.0695 + 0.01j, 1.0509
    M = dense_matrix(U, m, c_sw)
    b = synth.point_source(L, T, spin=2, colour=1)
    x_lu = np.linalg.solve(M, b.ravel())
    x, info = oracle.bicgstab(U, b, m, c_sw, tol=1e-13)
    assert info["status"] == 0 and info["true_resid"] < 1e-12
    assert rel(x.ravel(), x_lu) < 1e-11


def test_free_propagator_by_fourier_sum(gammas):
    """Free-field point-source propagator x(y) = (1/V) sum_p e^{i p y} D(p)^{-1} u with
    D(p) = sum_mu [cos p_mu + i g_mu sin p_mu] - (4 + Re m) - i Im m g5 (the Fourier transform of Eq. 2 at U = 1)."""
    L, T = 4, 8
    m = 0.1 + 0.05j
    spin, colour = 1, 2
    b = synth.point_source(L, T, spin=spin, colour=colour)
    x, info = oracle.bicgstab(synth.unit_gauge(L, T), b, m, tol=1e-13)
    assert info["status"] == 0
    g5 = gammas[0] @ gammas[1] @ gammas[2] @ gammas[3]
    xs, ys, zs, ts = coords(L, T)
    acc = np.zeros((T, L, L, L, 4), dtype=np.complex128)
    e = np.zeros(4, dtype=np.complex128)
    e[spin] = 1.0
    for n in itertools.product(range(L), range(L), range(L), range(T)):
        p = momentum(L, T, n)
        Dp = sum(np.cos(p[mu]) * np.eye(4) + 1j * np.sin(p[mu]) * gammas[mu] for mu in range(4))
        Dp = Dp - (4.0 + m.real) * np.eye(4) - 1j * m.imag * g5
        w = np.linalg.solve(Dp, e)
        phase = np.exp(1j * (p[0] * xs + p[1] * ys + p[2] * zs + p[3] * ts))
        acc += phase[..., None] * w
    acc /= L ** 3 * T
    expect = np.zeros_like(b)
    expect[..., colour] = acc
    assert rel(x, expect) < 1e-11


def test_config0_solves_in_seconds():
    """BASELINE.json configs[0]: 4^3 x 8, m = 0.1, no clover, eps = 0.3, seed 1, point source, tol 1e-10."""
    cfg = synth.CONFIGS[0]
    U = synth.gauge_field(cfg["L"], cfg["T"], cfg["eps"], seed=1)
    b = synth.point_source(cfg["L"], cfg["T"])
    x, info = oracle.bicgstab(U, b, complex(*cfg["m"]), cfg["c_sw"], tol=1e-10)
    assert info["status"] == 0 and info["true_resid"] <= 1e-10
    assert info["iters"] < 100


def test_zero_source_gives_zero_solution():
    U = synth.gauge_field(2, 2, 0.3, seed=1)
    x, info = oracle.bicgstab(U, np.zeros((2, 2, 2, 2, 4, 3), dtype=np.complex128), 0.1)
    assert info["status"] == 0 and np.all(x == 0)


def test_bicgstab_exact_at_the_half_step():
    """The <t,t> = 0 exit of the oracle's BiCGStab (s = r - alpha v vanished: x + alpha p is the solution). Without that exit
    omega = 0/0 poisons x; an exit that forgets x += alpha p returns 0. Closed form: D b = 2 b, so x = b / 2 after ONE
    iteration with a residual of exactly 0."""
    U, b = H.exact_eigenvector_case()
    assert np.array_equal(oracle.apply(U, b, -2.0), 2.0 * b)  # the premise, bit for bit
    x, info = oracle.bicgstab(U, b, -2.0, tol=1e-12)
    assert info["status"] == 0 and info["iters"] == 1 and info["true_resid"] == 0.0
    assert np.array_equal(x, 0.5 * b)


# ----------------------------------------------------------------------------------------------------------
# (e) gamma5 D and the Chebyshev series of it
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c_sw", [0.0, 1.1])
def test_gamma5_D_is_hermitian_for_real_mass(c_sw):
    """gamma5-hermiticity D^dag = g5 D g5 (pin (b)) makes H_w = g5 D Hermitian when m is real: <y, H x> = <H y, x>,
    and H^2 = D^dag D. A wrong gamma5 (sign, basis, acting on colour instead of spin) breaks one of the two."""
    L, T, m = 4, 4, -0.3
    U = synth.gauge_field(L, T, 0.4, seed=1)
    x, y = synth.gaussian_spinor(L, T, 3), synth.gaussian_spinor(L, T, 4)
    Hx, Hy = oracle.gamma5_apply(U, x, m, c_sw), oracle.gamma5_apply(U, y, m, c_sw)
    assert abs(vdot(y, Hx) - vdot(Hy, x)) <= 1e-12 * abs(vdot(y, Hx))
    HHx = oracle.gamma5_apply(U, Hx, m, c_sw)
    DdDx = oracle.apply(U, oracle.apply(U, x, m, c_sw), m, c_sw, dagger=True)
    assert rel(HHx, DdDx) <= 1e-13
    # gamma5 itself: diag(+1,+1,-1,-1) on the spin index (golden table, C5)
    assert np.array_equal(oracle.gamma5_apply(U, x, m, c_sw)[..., 2:, :], -oracle.apply(U, x, m, c_sw)[..., 2:, :])
    assert np.array_equal(oracle.gamma5_apply(U, x, m, c_sw)[..., :2, :], oracle.apply(U, x, m, c_sw)[..., :2, :])


def test_cheb_series_vs_eigendecomposition_2x2x2x2():
    """On 2^4 the Hermitian X = scale * g5 D + shift is a 192 x 192 matrix: sum_k c_k T_k(X) psi must equal
    V chebval(lambda, c) V^dag psi (numpy's Chebyshev evaluation on the eigenvalues). Pins the recurrence
    (T_{k+1} = 2 X T_k - T_{k-1}), the role of scale and shift, and the coefficient order."""
    L = T = 2
    m, c_sw = -0.2, 1.0
    U = synth.gauge_field(L, T, 0.4, seed=1)
    psi = synth.gaussian_spinor(L, T, 3)
    g5 = np.kron(np.eye(L ** 3 * T), np.kron(oracle.gamma(4), np.eye(3)))
    H = g5 @ dense_matrix(U, m, c_sw)
    assert np.linalg.norm(H - H.conj().T) <= 1e-12 * np.linalg.norm(H)
    lam = np.linalg.eigvalsh(H)
    scale, shift = 1.7 / (lam.max() - lam.min()), 0.05
    X = scale * H + shift * np.eye(H.shape[0])
    w, V = np.linalg.eigh(X)
    assert w.min() > -1 and w.max() < 1
    rng = np.random.default_rng(5)
    for n in (1, 2, 3, 12):
        coef = rng.standard_normal(n)
        ref = V @ (np.polynomial.chebyshev.chebval(w, coef) * (V.conj().T @ psi.ravel()))
        got = oracle.cheb_series(U, psi, coef, scale, shift, m, c_sw).ravel()
        assert rel(got, ref) <= 1e-12, n


def test_cheb_series_single_polynomials_free_field():
    """T_k(cos theta) = cos(k theta): on a free-field plane-wave eigenvector of H^2 = D^dag D ... use instead the
    exact operator identity T_2(X) = 2 X^2 - 1 and T_3(X) = 4 X^3 - 3 X on a random field."""
    L, T, m = 4, 4, 0.1
    U = synth.gauge_field(L, T, 0.3, seed=1)
    psi = synth.gaussian_spinor(L, T, 3)
    scale, shift = 0.2, -0.1
    X = lambda v: scale * oracle.gamma5_apply(U, v, m) + shift * v
    X1 = X(psi); X2 = X(X1); X3 = X(X2)
    assert rel(oracle.cheb_series(U, psi, [0, 0, 1.0], scale, shift, m), 2 * X2 - psi) <= 1e-13
    assert rel(oracle.cheb_series(U, psi, [0, 0, 0, 1.0], scale, shift, m), 4 * X3 - 3 * X1) <= 1e-13
