"""Parity of the CUDA path (libtmw.so through its C ABI) with the fp64 CPU oracle on identical seeded inputs.

Tolerances (BASELINE.json north_star):
  fp32 Dslash / Schur / clover: max over sites of |out_gpu(x) - out_ref(x)|_2 / |out_ref(x)|_2 <= 1e-5
  fp64 kernels:                 the same measure <= 1e-12 (rounding-order differences only)
  solves: fp64 true residual (recomputed by the ORACLE's operator) <= 1e-10, |x_gpu - x_oracle| / |x_oracle| <= 1e-8
  layout conversion: bit exact.
"""
import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL32, TOL64 = 1e-5, 1e-12


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()  # raises if libtmw.so is missing: no fallback
    return m


def dev(a: np.ndarray):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def packed_empty(ctx, tmw, prec):
    return torch.empty(ctx.spinor_bytes(prec), dtype=torch.uint8, device="cuda")


def gpu_pack(ctx, tmw, psi, par, prec):
    """canonical numpy spinor -> packed device buffer via the library's own tmw_pack"""
    d = dev(psi)
    out = packed_empty(ctx, tmw, prec)
    ctx.pack(prec, tmw.ODD if par else tmw.EVEN, d, out)
    torch.cuda.synchronize()
    return out


def gpu_unpack(ctx, tmw, packed, par, prec, L, T):
    out = torch.zeros((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
    ctx.unpack(prec, tmw.ODD if par else tmw.EVEN, packed, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def mask_parity(psi, par_keep):
    """copy of psi with the sites of the other parity zeroed"""
    T, L = psi.shape[0], psi.shape[1]
    out = psi.copy().reshape(-1, 12)
    out[H.parity_sites(L, T, 1 - par_keep)] = 0
    return out.reshape(psi.shape)


def site_matrices(U, m, c_sw, dagger=False, mass_scalar=False):
    """A(x) as (V,12,12) from the oracle: apply D to vectors supported on one parity and read the same parity."""
    T, L = U.shape[1], U.shape[2]
    V = L ** 3 * T
    F = oracle.field_strength(U) if c_sw != 0 else None
    A = np.zeros((V, 12, 12), dtype=np.complex128)
    for par in (0, 1):
        s = H.parity_sites(L, T, par)
        for k in range(12):
            e = np.zeros((V, 12), dtype=np.complex128)
            e[s, k] = 1.0
            col = oracle.apply(U, e.reshape(T, L, L, L, 4, 3), m, c_sw, dagger=dagger, F=F,
                               mass_reading=int(mass_scalar)).reshape(V, 12)
            A[s, :, k] = col[s]
    return A


# ------------------------------------------------------------------------------------------------------
# layout conversion (A0): bit exact against the numpy restatement of the layout in include/tmw.h
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,T", [(4, 8), (6, 4)])
def test_pack_unpack_bit_exact(tmw, L, T):
    U = synth.gauge_field(L, T, 0.3, seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    with tmw.Context(L, T, dev(U), 0.1) as ctx:
        for prec, dt in ((tmw.F32, np.float32), (tmw.F64, np.float64)):
            assert ctx.spinor_bytes(prec) == L ** 3 * T // 2 * 24 * np.dtype(dt).itemsize
            full = np.zeros_like(psi)
            for par in (0, 1):
                p = gpu_pack(ctx, tmw, psi, par, prec)
                got = p.cpu().numpy().view(dt)
                ref = H.pack_spinor(psi, par, dt)
                assert np.array_equal(got, ref.ravel())
                back = gpu_unpack(ctx, tmw, p, par, prec, L, T)
                full += back
                assert np.array_equal(mask_parity(back, par), back)
            assert np.array_equal(full, psi.astype(np.complex64 if dt == np.float32 else np.complex128).astype(np.complex128))


# ------------------------------------------------------------------------------------------------------
# the hopping stencil H_{p pbar} (A3), every (op, parity, precision, reconstruct) combination
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,T,eps", [(4, 8, 0.3), (6, 4, 0.4), (8, 16, 0.4), (12, 10, 0.35)])
def test_hopping_vs_oracle(tmw, L, T, eps):
    U = synth.gauge_field(L, T, eps, seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    z2 = synth.z2_source(L, T, seed=2)
    for recon in (12, 18):
        with tmw.Context(L, T, dev(U), 0.1, reconstruct=recon) as ctx:
            for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
                if prec == tmw.F64 and recon == 18:
                    continue  # the fp64 path always stores 18 reals: covered by recon = 12
                for src in (psi, z2):
                    for op in (tmw.D, tmw.DDAG):
                        for par in (0, 1):
                            inp = gpu_pack(ctx, tmw, src, 1 - par, prec)
                            out = packed_empty(ctx, tmw, prec)
                            ctx.apply(op, tmw.ODD if par else tmw.EVEN, prec, inp, out)
                            got = gpu_unpack(ctx, tmw, out, par, prec, L, T)
                            # oracle: D on the source masked to parity pbar; on parity p only the hopping term acts
                            ref = mask_parity(oracle.apply(U, mask_parity(src, 1 - par), 0.1, dagger=(op == tmw.DDAG)), par)
                            site, glob = H.per_site_rel_err(got, ref)
                            assert site <= tol, (recon, prec, op, par, site, glob)


def test_hopping_point_source_exact_zeros(tmw):
    """C16: sites the stencil does not reach must be exactly zero (point source at the origin)."""
    L, T = 4, 8
    U = synth.gauge_field(L, T, 0.3, seed=1)
    b = synth.point_source(L, T, 0, 0)
    with tmw.Context(L, T, dev(U), 0.1) as ctx:
        inp = gpu_pack(ctx, tmw, b, 0, tmw.F32)
        out = packed_empty(ctx, tmw, tmw.F32)
        ctx.apply(tmw.D, tmw.ODD, tmw.F32, inp, out)
        got = gpu_unpack(ctx, tmw, out, 1, tmw.F32, L, T)
        ref = mask_parity(oracle.apply(U, b, 0.1), 1)
        site, _ = H.per_site_rel_err(got, ref)  # asserts exact zeros where ref == 0
        assert site <= TOL32
        assert np.count_nonzero(np.abs(got).sum(axis=(-1, -2))) == 8


# ------------------------------------------------------------------------------------------------------
# full operator (A3 + A4): mass, twist (both readings), clover, D and D^dagger
# ------------------------------------------------------------------------------------------------------
CASES_FULL = [
    dict(L=4, T=8, eps=0.3, m=0.1 + 0.0j, c_sw=0.0),
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0),
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.25j, c_sw=0.0, scalar=True),
    dict(L=4, T=6, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509),
    dict(L=8, T=6, eps=0.35, m=-0.0514 + 0.0j, c_sw=1.0424),
    dict(L=4, T=6, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349),
]


@pytest.mark.parametrize("case", CASES_FULL)
def test_full_apply_vs_oracle(tmw, case):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    scalar = case.get("scalar", False)
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    rd = tmw.MASS_SCALAR if scalar else tmw.TWIST_GAMMA5
    with tmw.Context(L, T, dev(U), m, c_sw, mass_reading=rd) as ctx:
        for op in (tmw.D, tmw.DDAG):
            out = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
            ctx.apply(op, tmw.FULL, tmw.F64, dev(psi), out)
            torch.cuda.synchronize()
            ref = oracle.apply(U, psi, m, c_sw, dagger=(op == tmw.DDAG), mass_reading=int(scalar))
            site, glob = H.per_site_rel_err(out.cpu().numpy(), ref)
            assert site <= TOL64, (op, site, glob)
    # HOST location: numpy arrays straight through the C ABI
    with tmw.Context(L, T, U, m, c_sw, mass_reading=rd, location=tmw.HOST) as ctx:
        out = np.empty_like(psi)
        ctx.apply(tmw.D, tmw.FULL, tmw.F64, psi, out)
        site, _ = H.per_site_rel_err(out, oracle.apply(U, psi, m, c_sw, mass_reading=int(scalar)))
        assert site <= TOL64


@pytest.mark.parametrize("L,T", [(8, 6), (8, 16), (8, 4), (16, 4)])
def test_full_apply_host_pipelined_vs_oracle(tmw, L, T):
    """tmw_apply FULL with HOST pointers on lattices whose time slices are multiples of 128 checkerboard sites: the path that
    cuts the spinor into t-slabs and overlaps upload, operator and download on three streams (T = 6: 6 slabs, 16: 8 slabs
    of 2, 4: 4 slabs of 1). D, D^dag and gamma5 D, pinned and pageable host memory, twice in a row (buffer reuse)."""
    m, c_sw = -0.0514 + 0.02j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    psi = synth.gaussian_spinor(L, T, seed=3)
    with tmw.Context(L, T, U, m, c_sw, location=tmw.HOST) as ctx:
        for rep in range(2):
            for op in (tmw.D, tmw.DDAG, tmw.G5D):
                src = torch.from_numpy(psi).pin_memory() if rep else psi
                out = np.full_like(psi, 7.0)
                ctx.apply(op, tmw.FULL, tmw.F64, src.data_ptr() if rep else src, out)
                ref = oracle.gamma5_apply(U, psi, m, c_sw, F=F) if op == tmw.G5D else oracle.apply(U, psi, m, c_sw, dagger=(op == tmw.DDAG), F=F)
                site, _ = H.per_site_rel_err(out, ref)
                assert site <= TOL64, (rep, op, site)


# ------------------------------------------------------------------------------------------------------
# clover blocks (A1) and their inverse (A2) against the oracle's F and sigma
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pivot,reconstruct", [(False, 12), (True, 12), (False, 18)])
@pytest.mark.parametrize("L,T,m,c_sw", [(4, 6, -0.0695 + 0.0j, 1.0509), (6, 4, -0.044 + 0.2j, 1.0349), (8, 4, -3.9 + 0.0j, 2.5)])
def test_clover_blocks_and_inverse(tmw, L, T, m, c_sw, pivot, reconstruct):
    """the third case makes the blocks indefinite (diagonal -(4+m) = -0.1, clover term of order 1): the unpivoted
    L D L^dag still has to invert them; pivot = True forces the Gauss-Jordan fallback kernel (TMW_DEBUG_FORCE_PIVOT).
    reconstruct = 12: the plaquette products rebuild their third row from the first two (SU(3) links); 18: all three rows
    are multiplied out."""
    U = synth.gauge_field(L, T, 0.4, seed=1)
    blocks = H.site_diagonal_blocks(U, c_sw, m.real)  # (V,2,6,6)
    Vh = L ** 3 * T // 2
    with tmw.Context(L, T, dev(U), m, c_sw, debug=tmw.DEBUG_FORCE_PIVOT if pivot else 0, reconstruct=reconstruct) as ctx:
        for par in (0, 1):
            dst = torch.empty((Vh, 2, 36), dtype=torch.float64, device="cuda")
            ctx.get_clover(tmw.ODD if par else tmw.EVEN, 0, dst)
            torch.cuda.synchronize()
            ref = H.pack_hermitian(blocks[H.parity_sites(L, T, par)])
            assert np.max(np.abs(dst.cpu().numpy() - ref)) <= 1e-13
        dst = torch.empty((Vh, 2, 36), dtype=torch.float64, device="cuda")
        ctx.get_clover(tmw.EVEN, 1, dst)
        torch.cuda.synchronize()
        be = blocks[H.parity_sites(L, T, 0)]
        ref_inv = np.linalg.inv(be @ be + m.imag ** 2 * np.eye(6)) if m.imag != 0 else np.linalg.inv(be)
        ref = H.pack_hermitian(ref_inv)
        got = dst.cpu().numpy()
        # relative to each block's own largest entry (indefinite blocks can have large inverses)
        scale = np.max(np.abs(ref), axis=-1, keepdims=True)
        cond = np.linalg.cond(be @ be + m.imag ** 2 * np.eye(6) if m.imag != 0 else be)
        assert np.max(np.abs(got - ref) / scale / cond[..., None]) <= 1e-13


# ------------------------------------------------------------------------------------------------------
# Schur complement (A5 = K1 then K2) in fp32 and fp64 against the oracle's masked pieces
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", [
    dict(L=4, T=8, eps=0.3, m=0.1 + 0.0j, c_sw=0.0),
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0),
    dict(L=4, T=6, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509),
    dict(L=4, T=6, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349),
])
def test_schur_vs_oracle(tmw, case):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    V = L ** 3 * T
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    F = oracle.field_strength(U) if c_sw != 0 else None
    ev, od = H.parity_sites(L, T, 0), H.parity_sites(L, T, 1)
    with tmw.Context(L, T, dev(U), m, c_sw) as ctx:
        for op in (tmw.D, tmw.DDAG):
            dag = op == tmw.DDAG
            A = site_matrices(U, m, c_sw, dagger=dag)
            x_o = mask_parity(psi, 1)
            Dx = oracle.apply(U, x_o, m, c_sw, dagger=dag, F=F).reshape(V, 12)  # even: H_eo x_o; odd: A_oo x_o
            t_e = np.zeros((V, 12), dtype=np.complex128)
            t_e[ev] = np.linalg.solve(A[ev], Dx[ev][..., None])[..., 0]
            Dt = oracle.apply(U, t_e.reshape(psi.shape), m, c_sw, dagger=dag, F=F).reshape(V, 12)  # odd: H_oe t_e
            ref = np.zeros((V, 12), dtype=np.complex128)
            ref[od] = Dx[od] - Dt[od]
            for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
                inp = gpu_pack(ctx, tmw, psi, 1, prec)
                out = packed_empty(ctx, tmw, prec)
                ctx.apply_schur(op, prec, inp, out)
                got = gpu_unpack(ctx, tmw, out, 1, prec, L, T)
                site, glob = H.per_site_rel_err(got, ref.reshape(psi.shape))
                assert site <= tol, (op, prec, site, glob)


# ------------------------------------------------------------------------------------------------------
# solves (A5-A8)
# ------------------------------------------------------------------------------------------------------
def check_solution(U, b, x, m, c_sw, x_ref=None, mass_scalar=False, F=None):
    r = b - oracle.apply(U, x, m, c_sw, F=F, mass_reading=int(mass_scalar))
    resid = np.linalg.norm(r.ravel()) / np.linalg.norm(b.ravel())
    assert resid <= 1e-10, resid
    if x_ref is not None:
        err = np.linalg.norm((x - x_ref).ravel()) / np.linalg.norm(x_ref.ravel())
        assert err <= 1e-8, err
    return resid


@pytest.mark.parametrize("precision", ["mixed", "double"])
def test_solve_exact_at_the_half_step(tmw, precision):
    """A source that is an eigenvector of D, set up so that no rounding error occurs (helpers.exact_eigenvector_case; the
    oracle's side of it is pinned in test_oracle_pins.py): s = r - alpha v vanishes identically, <t,t> = 0, and the guard in
    sc_omega_kernel (omega = beta = 0 instead of 0/0) has to carry the solve to x = b / 2. Links with det = -1: 18-real."""
    L, T, m = 4, 8, -2.0 + 0.0j
    U, b = H.exact_eigenvector_case(L, T)
    x_ref, oinfo = oracle.bicgstab(U, b, m, tol=1e-12)
    assert oinfo["status"] == 0 and oinfo["iters"] == 1
    with tmw.Context(L, T, dev(U), m, 0.0, reconstruct=18, precision=tmw.MIXED if precision == "mixed" else tmw.DOUBLE) as ctx:
        x = torch.full(b.shape, float("nan"), dtype=torch.complex128, device="cuda")
        info = ctx.solve(dev(b), x, 1e-10)
        x = x.cpu().numpy()
    assert np.all(np.isfinite(x)), info
    assert info["iters"] <= 2 and info["true_resid"] <= 1e-10, info
    check_solution(U, b, x, m, 0.0, x_ref)


SOLVE_CASES = [
    dict(L=4, T=8, eps=0.3, m=0.1 + 0.0j, c_sw=0.0, src="point"),           # BASELINE.json configs[0]
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0, src="z2"),         # configs[1] parameters, small
    dict(L=4, T=6, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509, src="point"),    # configs[2] parameters, small
    dict(L=6, T=8, eps=0.3, m=-0.044 + 0.005j, c_sw=1.0349, src="gauss"),   # Table 2 row 4: twist + clover
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.25j, c_sw=0.0, src="z2", scalar=True),
]


def make_source(case):
    L, T = case["L"], case["T"]
    return {"point": lambda: synth.point_source(L, T, 0, 0), "z2": lambda: synth.z2_source(L, T, 2),
            "gauss": lambda: synth.gaussian_spinor(L, T, 3)}[case["src"]]()


@pytest.mark.parametrize("precision", ["mixed", "double"])
@pytest.mark.parametrize("case", SOLVE_CASES)
def test_solve_vs_oracle(tmw, case, precision):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    scalar = case.get("scalar", False)
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    b = make_source(case)
    x_ref, info_ref = oracle.bicgstab(U, b, m, c_sw, tol=1e-12, mass_reading=int(scalar))
    assert info_ref["status"] == 0 and info_ref["true_resid"] < 1e-11
    with tmw.Context(L, T, dev(U), m, c_sw, precision=tmw.MIXED if precision == "mixed" else tmw.DOUBLE,
                     mass_reading=tmw.MASS_SCALAR if scalar else tmw.TWIST_GAMMA5) as ctx:
        x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        info = ctx.solve(dev(b), x, 1e-10)
        assert info["true_resid"] <= 1e-10 and info["iters"] > 0
        check_solution(U, b, x.cpu().numpy(), m, c_sw, x_ref, mass_scalar=scalar)


def test_solve_host_pointers_and_12_columns(tmw):
    """configs[3] shape of work (12 point sources one after another, C13) on a small lattice, HOST location."""
    L, T, m, c_sw = 4, 6, -0.0514 + 0.0j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    with tmw.Context(L, T, U, m, c_sw, location=tmw.HOST) as ctx:
        for spin in range(4):
            for colour in range(3):
                b = synth.point_source(L, T, spin, colour)
                x = np.empty_like(b)
                info = ctx.solve(b, x, 1e-10)
                assert info["true_resid"] <= 1e-10
                x_ref, _ = oracle.bicgstab(U, b, m, c_sw, tol=1e-12, F=F)
                check_solution(U, b, x, m, c_sw, x_ref, F=F)


def test_solve_edge_cases(tmw):
    L, T = 4, 4
    U = synth.gauge_field(L, T, 0.3, seed=1)
    b = synth.gaussian_spinor(L, T, 3)
    with tmw.Context(L, T, dev(U), 0.1, max_iter=2) as ctx:
        x = torch.full((T, L, L, L, 4, 3), 7.0, dtype=torch.complex128, device="cuda")
        # b = 0 -> x = 0
        info = ctx.solve(torch.zeros_like(x), x, 1e-10)
        assert info["iters"] == 0 and torch.count_nonzero(x).item() == 0
        # max_iter reached -> ENOCONV, x holds the best iterate (a reduced residual), info filled
        info = ctx.solve(dev(b), x, 1e-10, allow_noconv=True)
        assert info["status"] == tmw.ENOCONV and info["iters"] == 2
        assert 1e-10 < info["true_resid"] < 1.0
        r = b - oracle.apply(U, x.cpu().numpy(), 0.1)
        assert abs(np.linalg.norm(r.ravel()) / np.linalg.norm(b.ravel()) - info["true_resid"]) < 1e-9
        with pytest.raises(tmw.TmwError) as e:
            ctx.solve(dev(b), x, 0.0)
        assert e.value.code == tmw.EINVAL
        with pytest.raises(tmw.TmwError) as e:
            ctx.solve(x, x, 1e-10)
        assert e.value.code == tmw.EINVAL


def test_create_errors(tmw):
    U = dev(synth.gauge_field(4, 4, 0.3, seed=1))
    for L, T in ((3, 4), (4, 5), (2, 4)):
        with pytest.raises(tmw.TmwError) as e:
            tmw.Context(L, T, U, 0.1)
        assert e.value.code == tmw.EINVAL
    with pytest.raises(tmw.TmwError) as e:
        tmw.Context(4, 4, U, 0.1, reconstruct=13)
    assert e.value.code == tmw.EINVAL
    with pytest.raises(tmw.TmwError) as e:
        tmw.Context(4, 4, U, -4.0)  # 4 + m = 0: singular diagonal
    assert e.value.code == tmw.ESINGULAR
    # unit gauge: F = 0, the clover block is -(4+m) = 0 -> singular clover inverse
    with pytest.raises(tmw.TmwError) as e:
        tmw.Context(4, 4, dev(synth.unit_gauge(4, 4)), -4.0, 1.0)
    assert e.value.code == tmw.ESINGULAR


def test_solve_hard_system_with_restarts(tmw):
    """A smooth field close to the critical mass (eps = 0.1, m = -0.2, c_sw = 1): BiCGStab needs hundreds of iterations
    and its <rhat, r> decays to the noise several times, so the restart path (rhat := r from the fp64 true residual,
    C11) is exercised; restarts are allowed as long as they keep paying. Checked through the oracle's operator."""
    L, T, m, c_sw = 8, 16, -0.2 + 0.0j, 1.0
    U = synth.gauge_field(L, T, 0.1, seed=1)
    b = synth.gaussian_spinor(L, T, 3)
    F = oracle.field_strength(U)
    sols = {}
    for precision in (tmw.MIXED, tmw.DOUBLE):
        with tmw.Context(L, T, dev(U), m, c_sw, precision=precision, max_iter=4000) as ctx:
            x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
            info = ctx.solve(dev(b), x, 1e-10)
            assert info["true_resid"] <= 1e-10 and info["iters"] > 100 and info["restarts"] >= 1, info
            sols[precision] = x.cpu().numpy()
            check_solution(U, b, sols[precision], m, c_sw, F=F)
    d = np.linalg.norm((sols[tmw.MIXED] - sols[tmw.DOUBLE]).ravel()) / np.linalg.norm(sols[tmw.DOUBLE].ravel())
    assert d <= 1e-6, d  # both have residual 1e-10; the condition number of this system is ~1e3
