"""Seeded input generators: structure of the synthetic fields."""
import numpy as np

from paper_2201_09004_b200 import synth


def test_links_are_su3_and_deterministic():
    U = synth.gauge_field(4, 8, 0.3, seed=1)
    assert U.shape == (4, 8, 4, 4, 4, 3, 3)
    UUd = np.einsum("...ab,...cb->...ac", U, U.conj())
    assert np.max(np.abs(UUd - np.eye(3))) < 1e-14
    assert np.max(np.abs(np.linalg.det(U) - 1.0)) < 1e-13
    # third row is exactly conj(row0 x row1): the 12-real reconstruction is exact in fp64
    r2 = np.conj(np.cross(U[..., 0, :], U[..., 1, :]))
    assert np.max(np.abs(r2 - U[..., 2, :])) < 1e-15
    assert np.array_equal(U, synth.gauge_field(4, 8, 0.3, seed=1))
    assert not np.array_equal(U, synth.gauge_field(4, 8, 0.3, seed=2))


def test_link_is_matrix_exponential_of_gell_mann_sum():
    """eps -> 0: U ~ 1 + i eps H with H traceless Hermitian of the stated normalisation: <|H_ab|^2> summed = 2*8."""
    eps = 1e-6  # second-order term eps*H^2/2 ~ 1e-5, rounding 1e-16/eps ~ 1e-10
    U = synth.su3_matrices(20000, eps, seed=5)
    H = (U - np.eye(3)) / (1j * eps)
    assert np.max(np.abs(H - np.conj(np.swapaxes(H, -1, -2)))) < 1e-3
    assert abs(np.mean(np.abs(np.trace(H, axis1=-2, axis2=-1)))) < 1e-3
    # tr(H^2) = 2 sum c_a^2, E = 16
    trh2 = np.real(np.einsum("nab,nba->n", H, H)).mean()
    assert abs(trh2 - 16.0) < 0.4


def test_plaquette_roughness():
    """The recipe gives rough fields (mean plaquette ~0.37 at eps = 0.3, ~0.16 at eps = 0.4)."""
    def plaq(U):
        acc, n = 0.0, 0
        for mu in range(4):
            for nu in range(mu + 1, 4):
                a = U[mu]
                b = np.roll(U[nu], -1, axis=3 - mu)
                c = np.roll(U[mu], -1, axis=3 - nu)
                d = U[nu]
                p = np.einsum("...ab,...bc,...dc,...ed->...ae", a, b, c.conj(), d.conj())
                acc += np.real(np.trace(p, axis1=-2, axis2=-1)).mean() / 3.0
                n += 1
        return acc / n
    p3 = plaq(synth.gauge_field(6, 6, 0.3, seed=1))
    p4 = plaq(synth.gauge_field(6, 6, 0.4, seed=1))
    assert 0.25 < p3 < 0.5 and 0.08 < p4 < 0.3 and p4 < p3


def test_sources():
    z = synth.z2_source(4, 4, seed=2)
    assert set(np.unique(z.real)) == {-1.0, 1.0} and np.all(z.imag == 0)
    assert abs(z.real.mean()) < 0.1
    g = synth.gaussian_spinor(6, 6, seed=3)
    assert abs(g.real.std() - 1) < 0.05 and abs(g.imag.std() - 1) < 0.05 and abs(g.mean()) < 0.05
    b = synth.point_source(4, 8, spin=2, colour=1, site=(1, 2, 3, 4))
    assert b.sum() == 1.0 and b[4, 3, 2, 1, 2, 1] == 1.0
