"""Parity of the multi-right-hand-side calls (tmw_apply_multi / tmw_apply_schur_multi / tmw_solve_multi, SURVEY §8(f1):
the "12 columns" of PAPER.md:78) with the fp64 CPU oracle, column by column, on identical seeded inputs.

The oracle has no multi-column notion: each column is an independent application / solve of the same operator, so the
expected values are the single-column oracle results. Tolerances as in test_gpu_parity.py.
"""
import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth
from test_gpu_parity import TOL32, TOL64, check_solution, dev, mask_parity, site_matrices

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()
    return m


TILES = {None: (0, 0, 0, 0), "auto": (-1, 0, 0, 0), "1,2,1,3": (1, 2, 1, 3)}
# columns per thread of the fp32 stencil (tmw_options.columns_per_thread)
SPREADS = [dict(columns_per_thread=n) for n in (1, 2, 3, 4)]


def columns(L, T, n):
    """n dense spinors with different seeds (Gaussian, every third one Z2)"""
    return [synth.z2_source(L, T, seed=100 + c) if c % 3 == 2 else synth.gaussian_spinor(L, T, seed=10 + c) for c in range(n)]


def pack_multi(ctx, tmw, cols, par, prec):
    nb = ctx.spinor_bytes(prec)
    buf = torch.empty(nb * len(cols), dtype=torch.uint8, device="cuda")
    for c, psi in enumerate(cols):
        ctx.pack(prec, tmw.ODD if par else tmw.EVEN, dev(psi), buf[c * nb:(c + 1) * nb])
    torch.cuda.synchronize()
    return buf


def unpack_multi(ctx, tmw, buf, n, par, prec, L, T):
    nb = ctx.spinor_bytes(prec)
    out = []
    for c in range(n):
        o = torch.zeros((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        ctx.unpack(prec, tmw.ODD if par else tmw.EVEN, buf[c * nb:(c + 1) * nb], o)
        out.append(o)
    torch.cuda.synchronize()
    return [o.cpu().numpy() for o in out]


@pytest.mark.parametrize("spread", SPREADS, ids=lambda d: "-".join(f"{k[8:]}{v}" for k, v in d.items()))
@pytest.mark.parametrize("L,T,nrhs,tile", [(8, 16, 5, "auto"), (8, 16, 5, None), (6, 4, 12, None), (4, 8, 7, "auto"), (4, 8, 3, "1,2,1,3")])
def test_hopping_multi_vs_oracle(tmw, L, T, nrhs, tile, spread):
    # tile: 4-D tiles of 128 sites instead of 128 consecutive checkerboard indices
    U = synth.gauge_field(L, T, 0.4, seed=1)
    cols = columns(L, T, nrhs)
    with tmw.Context(L, T, dev(U), 0.1, tile=TILES[tile], **spread) as ctx:
        for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
            if prec == tmw.F64 and spread != SPREADS[0]:
                continue  # the fp64 stencil always takes one column per thread
            for op in (tmw.D, tmw.DDAG):
                for par in (0, 1):
                    inp = pack_multi(ctx, tmw, cols, 1 - par, prec)
                    out = torch.full_like(inp, 0x7f)
                    ctx.apply_multi(op, tmw.ODD if par else tmw.EVEN, prec, nrhs, inp, out)
                    got = unpack_multi(ctx, tmw, out, nrhs, par, prec, L, T)
                    for c in range(nrhs):
                        ref = mask_parity(oracle.apply(U, mask_parity(cols[c], 1 - par), 0.1, dagger=(op == tmw.DDAG)), par)
                        site, glob = H.per_site_rel_err(got[c], ref)
                        assert site <= tol, (prec, op, par, c, site, glob)


@pytest.mark.parametrize("L,T,nrhs,zchunk,cpt", [(8, 6, 5, 4, 2), (8, 4, 3, 4, 3), (16, 4, 2, 2, 2), (16, 4, 4, 8, 4), (8, 4, 2, 3, 2), (8, 4, 2, -1, 2)])
def test_zchunk_sweep_vs_oracle(tmw, L, T, nrhs, zchunk, cpt):
    """tmw_options.zchunk: the multi-column launches visit the site blocks slab by slab in z (all time slices of a slab
    first) - a permutation of the CTAs that must not change any output site. zchunk = 3 does not divide L (ignored)."""
    U = synth.gauge_field(L, T, 0.4, seed=1)
    cols = columns(L, T, nrhs)
    with tmw.Context(L, T, dev(U), 0.1, zchunk=zchunk, columns_per_thread=cpt) as ctx:
        for op in (tmw.D, tmw.DDAG):
            for par in (0, 1):
                inp = pack_multi(ctx, tmw, cols, 1 - par, tmw.F32)
                out = torch.full_like(inp, 0x7f)
                ctx.apply_multi(op, tmw.ODD if par else tmw.EVEN, tmw.F32, nrhs, inp, out)
                got = unpack_multi(ctx, tmw, out, nrhs, par, tmw.F32, L, T)
                for c in range(nrhs):
                    ref = mask_parity(oracle.apply(U, mask_parity(cols[c], 1 - par), 0.1, dagger=(op == tmw.DDAG)), par)
                    site, glob = H.per_site_rel_err(got[c], ref)
                    assert site <= TOL32, (op, par, c, site, glob)


@pytest.mark.parametrize("prefetch,nrhs,zchunk", [(1, 4, 0), (5, 3, 4), (1000, 2, 0), (3, 1, 0), (-1, 4, 0)])
def test_link_prefetch_changes_nothing(tmw, prefetch, nrhs, zchunk):
    """tmw_options.prefetch: prefetch.global.L2 of the links of a later site block (also past the end of the lattice) is a
    hint: hop and K1 / K2 outputs against the oracle as without it"""
    L, T, m, c_sw = 8, 4, -0.0695 + 0.0j, 1.0509
    U = synth.gauge_field(L, T, 0.4, seed=1)
    cols = columns(L, T, nrhs)
    F = oracle.field_strength(U)
    with tmw.Context(L, T, dev(U), m, c_sw, prefetch=prefetch, zchunk=zchunk) as ctx:
        inp = pack_multi(ctx, tmw, cols, 0, tmw.F32)
        out = torch.full_like(inp, 0x7f)
        ctx.apply_multi(tmw.D, tmw.ODD, tmw.F32, nrhs, inp, out)
        got = unpack_multi(ctx, tmw, out, nrhs, 1, tmw.F32, L, T)
        for c in range(nrhs):
            ref = mask_parity(oracle.apply(U, mask_parity(cols[c], 0), m, 0.0), 1)
            assert H.per_site_rel_err(got[c], ref)[0] <= TOL32, c
        b = np.stack([synth.point_source(L, T, c % 4, c % 3) for c in range(nrhs)])
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(nrhs, dev(b), x, 1e-10)
        x = x.cpu().numpy()
        for c in range(nrhs):
            assert infos[c]["true_resid"] <= 1e-10
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)


@pytest.mark.parametrize("zchunk,cpt", [(4, 2), (4, 3), (-1, 4)])
def test_zchunk_solve_vs_oracle(tmw, zchunk, cpt):
    """the z-slab sweep under K1, K2 and their fused dot products: 8^3 x 4 clover, six columns through tmw_solve_multi"""
    L, T, m, c_sw = 8, 4, -0.0514 + 0.0j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    b = np.stack([synth.point_source(L, T, c // 3, c % 3) for c in (0, 2, 5, 7, 9, 11)])
    with tmw.Context(L, T, dev(U), m, c_sw, zchunk=zchunk, columns_per_thread=cpt) as ctx:
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(6, dev(b), x, 1e-10)
        x = x.cpu().numpy()
        for c in range(6):
            assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)


@pytest.mark.parametrize("spread", SPREADS[1:], ids=lambda d: "-".join(f"{k[8:]}{v}" for k, v in d.items()))
@pytest.mark.parametrize("case", [
    dict(L=8, T=4, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509, nrhs=5),
    dict(L=4, T=6, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349, nrhs=4),   # twisted clover: two-factor inverse
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0, nrhs=12),
])
def test_schur_multi_vs_oracle(tmw, case, spread):
    tile = TILES["auto"] if spread.get("columns_per_thread") == 3 else TILES[None]
    L, T, m, c_sw, nrhs = case["L"], case["T"], case["m"], case["c_sw"], case["nrhs"]
    V = L ** 3 * T
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    cols = columns(L, T, nrhs)
    F = oracle.field_strength(U) if c_sw != 0 else None
    ev, od = H.parity_sites(L, T, 0), H.parity_sites(L, T, 1)
    A = site_matrices(U, m, c_sw)
    refs = []
    for psi in cols:
        Dx = oracle.apply(U, mask_parity(psi, 1), m, c_sw, F=F).reshape(V, 12)
        t_e = np.zeros((V, 12), dtype=np.complex128)
        t_e[ev] = np.linalg.solve(A[ev], Dx[ev][..., None])[..., 0]
        Dt = oracle.apply(U, t_e.reshape(psi.shape), m, c_sw, F=F).reshape(V, 12)
        ref = np.zeros((V, 12), dtype=np.complex128)
        ref[od] = Dx[od] - Dt[od]
        refs.append(ref.reshape(psi.shape))
    with tmw.Context(L, T, dev(U), m, c_sw, tile=tile, **spread) as ctx:
        for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
            inp = pack_multi(ctx, tmw, cols, 1, prec)
            out = torch.full_like(inp, 0x7f)
            ctx.apply_schur_multi(tmw.D, prec, nrhs, inp, out)
            got = unpack_multi(ctx, tmw, out, nrhs, 1, prec, L, T)
            for c in range(nrhs):
                site, glob = H.per_site_rel_err(got[c], refs[c])
                assert site <= tol, (prec, c, site, glob)


@pytest.mark.parametrize("precision,spread", [("mixed", {}), ("double", {}), ("mixed", dict(columns_per_thread=1)),
                                              ("mixed", dict(columns_per_thread=3))])
def test_solve_multi_12_columns_vs_oracle(tmw, precision, spread):
    """configs[3] shape of work on a small lattice: the 12 point sources of a propagator (C13) in ONE call."""
    L, T, m, c_sw = 4, 8, -0.0514 + 0.0j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    b = np.stack([synth.point_source(L, T, c // 3, c % 3) for c in range(12)])
    with tmw.Context(L, T, dev(U), m, c_sw, precision=tmw.MIXED if precision == "mixed" else tmw.DOUBLE, **spread) as ctx:
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(12, dev(b), x, 1e-10)
        x = x.cpu().numpy()
        for c in range(12):
            assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)


def test_solve_multi_mixed_columns_host(tmw):
    """columns of different kind (point, Z2, Gaussian, zero, a scaled copy) converge at different iterations: columns
    drop out of the launches one by one; HOST pointers; twisted mass without clover (configs[1] parameters)."""
    L, T, m = 8, 4, -0.0695 + 0.01j
    U = synth.gauge_field(L, T, 0.4, seed=1)
    g = synth.gaussian_spinor(L, T, 3)
    b = np.stack([synth.point_source(L, T, 0, 0), synth.z2_source(L, T, 2), g, np.zeros_like(g), 1e-3 * g,
                  synth.point_source(L, T, 3, 2), synth.gaussian_spinor(L, T, 4)])
    n = b.shape[0]
    with tmw.Context(L, T, U, m, 0.0, location=tmw.HOST) as ctx:
        x = np.full(b.shape, 7.0 + 0j)
        infos = ctx.solve_multi(n, b, x, 1e-10)
        assert infos[3]["iters"] == 0 and np.count_nonzero(x[3]) == 0
        for c in range(n):
            if c == 3:
                continue
            assert infos[c]["true_resid"] <= 1e-10
            x_ref, _ = oracle.bicgstab(U, b[c], m, 0.0, tol=1e-12)
            check_solution(U, b[c], x[c], m, 0.0, x_ref)
        # a single solve afterwards (smaller batch than the workspace) gives the same answer as column 0
        x0 = np.empty_like(b[0])
        ctx.solve(b[0], x0, 1e-10)
        assert np.linalg.norm((x0 - x[0]).ravel()) <= 1e-9 * np.linalg.norm(x[0].ravel())


@pytest.mark.parametrize("solver", ["bicgstab", "gcr"])
def test_defect_correction_of_a_subset_leaves_the_other_columns_alone(tmw, solver):
    """The fp64 defect-correction pass (full-lattice residual above tol although the Schur system converged) re-solves only
    the columns that missed; TMW_DEBUG_FORCE_DEFECT sends columns 1 and 3 of 5 through it. Every column, corrected or not,
    must still be the oracle's solution (the pass once zeroed the odd-site solution of the columns it did not re-solve)."""
    L, T, m, c_sw = 4, 8, -0.0514 + 0.003j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    b = np.stack([synth.point_source(L, T, 0, 0), synth.gaussian_spinor(L, T, 3), synth.z2_source(L, T, 2),
                  synth.point_source(L, T, 2, 1), synth.gaussian_spinor(L, T, 4)])
    n = b.shape[0]
    with tmw.Context(L, T, dev(U), m, c_sw, solver=tmw.GCR if solver == "gcr" else tmw.BICGSTAB, debug=tmw.DEBUG_FORCE_DEFECT) as ctx:
        x = torch.full(b.shape, 7.0, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(n, dev(b), x, 1e-10)
        assert ctx.kernel_counts()["sub_norm"] >= 2 * 2 * 2  # b - D x and x + e, two parities, two columns
        x = x.cpu().numpy()
        for c in range(n):
            assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0, (c, infos[c])
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)


def test_solve_multi_edge_cases(tmw):
    L, T = 4, 4
    U = synth.gauge_field(L, T, 0.3, seed=1)
    b = np.stack([synth.gaussian_spinor(L, T, 3), synth.gaussian_spinor(L, T, 5)])
    with tmw.Context(L, T, dev(U), 0.1, max_iter=2) as ctx:
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(2, dev(b), x, 1e-10, allow_noconv=True)
        for c in range(2):
            assert infos[c]["status"] == tmw.ENOCONV and infos[c]["iters"] == 2 and 1e-10 < infos[c]["true_resid"] < 1.0
            r = b[c] - oracle.apply(U, x[c].cpu().numpy(), 0.1)
            assert abs(np.linalg.norm(r.ravel()) / np.linalg.norm(b[c].ravel()) - infos[c]["true_resid"]) < 1e-9
        for bad in (0, 17):
            with pytest.raises(tmw.TmwError) as e:
                ctx.solve_multi(bad, dev(b), x, 1e-10)
            assert e.value.code == tmw.EINVAL
