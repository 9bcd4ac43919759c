"""Domain-decomposed contexts (the paper's multi-GPU dimension: PAPER.md:52, the "Nodes" columns of
Table 2 :71-76, :315): tmw_options.domains_z x domains_t sub-lattices on ONE GPU, each with its own packed fields; every
stencil application = face pack of projected half spinors -> one copy per face -> interior pass (overlapping the copies)
-> exterior pass on the cut sites. Every call must (i) match the fp64 CPU oracle at the usual tolerances and (ii) match the
same call on an undivided context to rounding (the hops through a cut are added in a different order, nothing else).
"""
import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth
from test_gpu_parity import TOL32, TOL64, check_solution, dev, mask_parity, site_matrices

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

# (domains_z, domains_t): 2 and 2 x 2 domains as the time / z / both directions are cut, and 4 slabs in t
GRIDS = [(1, 2), (2, 1), (2, 2), (1, 4)]


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()
    return m


def roundtrip(ctx, tmw, fn, psi, par_in, par_out, prec, L, T):
    """pack psi (parity par_in) with the context's own layout, run fn(packed_in, packed_out), unpack parity par_out"""
    nb = ctx.spinor_bytes(prec)
    pin = torch.empty(nb, dtype=torch.uint8, device="cuda")
    pout = torch.full((nb,), 0x7f, dtype=torch.uint8, device="cuda")
    ctx.pack(prec, tmw.ODD if par_in else tmw.EVEN, dev(psi), pin)
    fn(pin, pout)
    out = torch.zeros((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
    ctx.unpack(prec, tmw.ODD if par_out else tmw.EVEN, pout, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("pz,pt", GRIDS)
@pytest.mark.parametrize("L,T", [(8, 8), (4, 8)])
def test_dd_hopping_vs_oracle_and_undivided(tmw, L, T, pz, pt):
    """L = 4 with domains_z = 2 gives local z extent 2 (every site is on a cut, both z hops of a site are ghosts or not)."""
    U = synth.gauge_field(L, T, 0.4, seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    with tmw.Context(L, T, dev(U), 0.1, domains_z=pz, domains_t=pt) as dd, tmw.Context(L, T, dev(U), 0.1) as one:
        for prec, tol, rnd in ((tmw.F32, TOL32, 2e-6), (tmw.F64, TOL64, 1e-14)):
            for op in (tmw.D, tmw.DDAG):
                for par in (0, 1):
                    call = lambda c: roundtrip(c, tmw, lambda a, b: c.apply(op, tmw.ODD if par else tmw.EVEN, prec, a, b), psi, 1 - par, par, prec, L, T)
                    got, ref1 = call(dd), call(one)
                    ref = mask_parity(oracle.apply(U, mask_parity(psi, 1 - par), 0.1, dagger=(op == tmw.DDAG)), par)
                    site, glob = H.per_site_rel_err(got, ref)
                    assert site <= tol, (prec, op, par, site, glob)
                    site1, _ = H.per_site_rel_err(got, ref1)
                    assert site1 <= rnd, (prec, op, par, site1)


@pytest.mark.parametrize("pz,pt", GRIDS)
@pytest.mark.parametrize("case", [
    dict(L=8, T=8, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509),   # clover K1 / K2
    dict(L=4, T=8, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349),    # twisted clover (two-factor inverse)
    dict(L=8, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0),     # twisted mass, no clover
])
def test_dd_schur_and_full_operator_vs_oracle(tmw, case, pz, pt):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    if T // pt < 2 or (T // pt) % 2:
        pytest.skip("local t extent must be even")
    V = L ** 3 * T
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    F = oracle.field_strength(U) if c_sw != 0 else None
    ev, od = H.parity_sites(L, T, 0), H.parity_sites(L, T, 1)
    with tmw.Context(L, T, dev(U), m, c_sw, domains_z=pz, domains_t=pt) as dd, tmw.Context(L, T, dev(U), m, c_sw) as one:
        for op in (tmw.D, tmw.DDAG):
            dag = op == tmw.DDAG
            A = site_matrices(U, m, c_sw, dagger=dag)
            Dx = oracle.apply(U, mask_parity(psi, 1), m, c_sw, dagger=dag, F=F).reshape(V, 12)
            t_e = np.zeros((V, 12), dtype=np.complex128)
            t_e[ev] = np.linalg.solve(A[ev], Dx[ev][..., None])[..., 0]
            Dt = oracle.apply(U, t_e.reshape(psi.shape), m, c_sw, dagger=dag, F=F).reshape(V, 12)
            ref = np.zeros((V, 12), dtype=np.complex128)
            ref[od] = Dx[od] - Dt[od]
            ref = ref.reshape(psi.shape)
            for prec, tol, rnd in ((tmw.F32, TOL32, 3e-6), (tmw.F64, TOL64, 1e-13)):
                call = lambda c: roundtrip(c, tmw, lambda a, b: c.apply_schur(op, prec, a, b), psi, 1, 1, prec, L, T)
                got, ref1 = call(dd), call(one)
                site, glob = H.per_site_rel_err(got, ref)
                assert site <= tol, (op, prec, site, glob)
                assert H.per_site_rel_err(got, ref1)[0] <= rnd
        # the full operator (Eq. (2) + (3)) in fp64 on canonical spinors, and gamma5 D
        out = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        for op in (tmw.D, tmw.DDAG, tmw.G5D):
            dd.apply(op, tmw.FULL, tmw.F64, dev(psi), out)
            torch.cuda.synchronize()
            ref = oracle.gamma5_apply(U, psi, m, c_sw, F=F) if op == tmw.G5D else oracle.apply(U, psi, m, c_sw, dagger=(op == tmw.DDAG), F=F)
            assert H.per_site_rel_err(out.cpu().numpy(), ref)[0] <= TOL64, op


@pytest.mark.parametrize("pz,pt", GRIDS)
@pytest.mark.parametrize("precision", ["mixed", "double"])
def test_dd_solve_vs_oracle(tmw, pz, pt, precision):
    """tmw_solve on 2, 2 x 2 and 4 domains: true residual through the ORACLE's D <= 1e-10, solution vs the oracle's <= 1e-8,
    and vs the undivided solve <= 1e-9 (different rounding, same system)."""
    L, T, m, c_sw = 8, 8, -0.0514 + 0.0j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    b = synth.point_source(L, T, 2, 1)
    x_ref, iref = oracle.bicgstab(U, b, m, c_sw, tol=1e-12, F=F)
    assert iref["status"] == 0
    prec = tmw.MIXED if precision == "mixed" else tmw.DOUBLE
    with tmw.Context(L, T, dev(U), m, c_sw, precision=prec, domains_z=pz, domains_t=pt) as dd, tmw.Context(L, T, dev(U), m, c_sw, precision=prec) as one:
        x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        x1 = torch.empty_like(x)
        info = dd.solve(dev(b), x, 1e-10)
        one.solve(dev(b), x1, 1e-10)
        assert info["true_resid"] <= 1e-10 and info["iters"] > 0
        check_solution(U, b, x.cpu().numpy(), m, c_sw, x_ref, F=F)
        assert float(torch.linalg.vector_norm(x - x1) / torch.linalg.vector_norm(x1)) <= 1e-9


def test_dd_solve_multi_twisted_and_gcr(tmw):
    """three columns in one tmw_solve_multi call on 2 x 2 domains (twisted mass, no clover), HOST pointers; GCR on 2 domains"""
    L, T, m = 8, 8, -0.0695 + 0.01j
    U = synth.gauge_field(L, T, 0.4, seed=1)
    b = np.stack([synth.point_source(L, T, 0, 0), synth.z2_source(L, T, 2), synth.gaussian_spinor(L, T, 3)])
    with tmw.Context(L, T, U, m, 0.0, location=tmw.HOST, domains_z=2, domains_t=2) as ctx:
        x = np.zeros_like(b)
        infos = ctx.solve_multi(3, b, x, 1e-10)
        for c in range(3):
            assert infos[c]["true_resid"] <= 1e-10
            x_ref, _ = oracle.bicgstab(U, b[c], m, 0.0, tol=1e-12)
            check_solution(U, b[c], x[c], m, 0.0, x_ref)
    with tmw.Context(L, T, dev(U), m, 0.0, solver=tmw.GCR, domains_t=2) as ctx:
        xg = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        info = ctx.solve(dev(b[2]), xg, 1e-10)
        assert info["true_resid"] <= 1e-10
        x_ref, _ = oracle.bicgstab(U, b[2], m, 0.0, tol=1e-12)
        check_solution(U, b[2], xg.cpu().numpy(), m, 0.0, x_ref)


def test_dd_option_errors(tmw):
    U = synth.gauge_field(4, 8, 0.3, seed=1)
    for kw in (dict(domains_z=3), dict(domains_t=3), dict(domains_z=4), dict(domains_t=8), dict(domains_z=-1)):
        with pytest.raises(tmw.TmwError) as e:
            tmw.Context(4, 8, dev(U), 0.1, **kw)
        assert e.value.code == tmw.EINVAL
    with tmw.Context(4, 8, dev(U), 0.1, 1.0, domains_t=2) as ctx:
        dst = torch.empty((4 ** 3 * 8 // 2, 2, 36), dtype=torch.float64, device="cuda")
        with pytest.raises(tmw.TmwError) as e:
            ctx.get_clover(tmw.EVEN, 0, dst)
        assert e.value.code == tmw.EINVAL
