"""Parity of the shared-memory staged fp32 stencil (csrc/tmw_dslash_stage.cuh; BASELINE.json north_star subsystem (2),
"neighbour tiles staged through TMA/shared memory") with the fp64 CPU oracle, on identical seeded inputs.

tmw_options.stage = 1 routes every fp32 hop / K1 / K2 launch through the staged kernel; stage_tile forces tile shapes
that exercise each branch of its index arithmetic: tiles that span x (wrap inside the staged row) and tiles with an x
halo, tiles as large as the lattice in y or z (the halo rows are the tile's own rows), CTAs with idle lanes
(tile sites not a multiple of 32), 1-3 columns per thread with ragged column groups. Expected values are the
single-column oracle results, tolerances as in test_gpu_parity.py.
"""
import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth
from test_gpu_multi import columns, pack_multi, unpack_multi
from test_gpu_parity import TOL32, check_solution, dev, mask_parity, site_matrices

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()
    return m


def staged_launches(ctx, fn):
    """run fn() and return how many stencil column applications went through the staged kernel (tmw_kernel_counts,
    TMW_K_STAGED), after checking that these were ALL the fp32 stencil applications of the call"""
    before = ctx.kernel_counts()
    fn()
    after = ctx.kernel_counts()
    n = after["staged"] - before["staged"]
    assert n == sum(after[k] - before[k] for k in ("hop32", "k1_32", "k2_32", "k2_32_dots"))
    return n


@pytest.mark.parametrize("L,T,nrhs,tile,cpt", [
    (8, 4, 5, (0, 0, 0), 2),     # automatic tile, ragged last group
    (8, 4, 3, (0, 0, 0), 3),
    (8, 4, 1, (0, 0, 0), 0),     # a single column through the staged kernel
    (8, 4, 4, (4, 2, 4), 2),     # spans x
    (8, 4, 4, (2, 2, 2), 2),     # x halo, 8 active lanes of 32
    (8, 6, 2, (2, 4, 2), 1),     # x halo, one column per thread, two groups
    (8, 4, 3, (1, 8, 2), 3),     # one x/2 site per row; the tile covers y completely
    (6, 4, 7, (3, 2, 2), 3),     # L/2 odd, 12 active lanes
    (6, 4, 2, (1, 2, 2), 2),
    (4, 8, 6, (2, 4, 4), 2),     # the tile is a whole time slice: every halo row is one of its own rows
    (4, 8, 5, (1, 4, 2), 1),
])
def test_hopping_staged_vs_oracle(tmw, L, T, nrhs, tile, cpt):
    U = synth.gauge_field(L, T, 0.4, seed=1)
    cols = columns(L, T, nrhs)
    with tmw.Context(L, T, dev(U), 0.1, stage=1, stage_tile=tile, columns_per_thread=cpt) as ctx:
        for op in (tmw.D, tmw.DDAG, tmw.G5D):
            for par in (0, 1):
                inp = pack_multi(ctx, tmw, cols, 1 - par, tmw.F32)
                out = torch.full_like(inp, 0x7f)
                n = staged_launches(ctx, lambda: ctx.apply_multi(op, tmw.ODD if par else tmw.EVEN, tmw.F32, nrhs, inp, out))
                assert n == nrhs
                got = unpack_multi(ctx, tmw, out, nrhs, par, tmw.F32, L, T)
                for c in range(nrhs):
                    ref = mask_parity(oracle.apply(U, mask_parity(cols[c], 1 - par), 0.1, dagger=(op == tmw.DDAG)), par)
                    if op == tmw.G5D:
                        ref = ref * np.array([1, 1, -1, -1])[:, None]
                    site, glob = H.per_site_rel_err(got[c], ref)
                    assert site <= TOL32, (op, par, c, site, glob)


def test_stage_is_used_and_matches_plain_kernel(tmw):
    """the staged and the plain kernel sum the same hops in a different order: equal to fp32 rounding, not bit for bit;
    with stage = -1 the same call must not touch the staged path"""
    L, T, nrhs = 8, 8, 4
    U = synth.gauge_field(L, T, 0.4, seed=1)
    cols = columns(L, T, nrhs)
    res = {}
    for stage in (-1, 1):
        with tmw.Context(L, T, dev(U), -0.05, 1.1, stage=stage) as ctx:
            inp = pack_multi(ctx, tmw, cols, 1, tmw.F32)
            out = torch.full_like(inp, 0x7f)
            ctx.apply_schur_multi(tmw.D, tmw.F32, nrhs, inp, out)
            assert ctx.kernel_counts()["staged"] == (2 * nrhs if stage == 1 else 0)
            res[stage] = np.stack(unpack_multi(ctx, tmw, out, nrhs, 1, tmw.F32, L, T))
    d = np.linalg.norm((res[1] - res[-1]).ravel()) / np.linalg.norm(res[-1].ravel())
    assert 0 < d <= 1e-6, d


@pytest.mark.parametrize("cpt", [1, 2, 3])
@pytest.mark.parametrize("case", [
    dict(L=8, T=4, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509, nrhs=5, tile=(0, 0, 0)),
    dict(L=4, T=6, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349, nrhs=4, tile=(2, 2, 4)),   # twisted clover: two-factor inverse
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0, nrhs=6, tile=(3, 2, 6)),    # twisted mass, no clover
])
def test_schur_staged_vs_oracle(tmw, case, cpt):
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
    with tmw.Context(L, T, dev(U), m, c_sw, stage=1, stage_tile=case["tile"], columns_per_thread=cpt) as ctx:
        inp = pack_multi(ctx, tmw, cols, 1, tmw.F32)
        out = torch.full_like(inp, 0x7f)
        n = staged_launches(ctx, lambda: ctx.apply_schur_multi(tmw.D, tmw.F32, nrhs, inp, out))
        assert n == 2 * nrhs
        got = unpack_multi(ctx, tmw, out, nrhs, 1, tmw.F32, L, T)
        for c in range(nrhs):
            site, glob = H.per_site_rel_err(got[c], refs[c])
            assert site <= TOL32, (c, site, glob)


@pytest.mark.parametrize("c_sw,m", [(1.0424, -0.0514 + 0.0j), (0.0, -0.0695 + 0.01j)])
def test_solve_multi_staged_vs_oracle(tmw, c_sw, m):
    """the fused dot products of the staged K2 launches drive the BiCGStab recurrences: 12 point sources in one call"""
    L, T = 8, 4
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U) if c_sw else None
    b = np.stack([synth.point_source(L, T, c // 3, c % 3) for c in range(12)])
    with tmw.Context(L, T, dev(U), m, c_sw, stage=1) as ctx:
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(12, dev(b), x, 1e-10)
        x = x.cpu().numpy()
        for c in range(12):
            assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)


def test_stage_bad_options(tmw):
    U = synth.gauge_field(4, 4, 0.3, seed=1)
    for kw in (dict(stage=2), dict(stage=-2), dict(stage_tile=(-1, 2, 2))):
        with pytest.raises(tmw.TmwError) as e:
            tmw.Context(4, 4, dev(U), 0.1, **kw)
        assert e.value.code == tmw.EINVAL
    # a tile that does not divide the lattice: the plain kernel runs, the result is unchanged
    psi = synth.gaussian_spinor(4, 4, seed=3)
    with tmw.Context(4, 4, dev(U), 0.1, stage=1, stage_tile=(2, 3, 2)) as ctx:
        inp = pack_multi(ctx, tmw, [psi], 0, tmw.F32)
        out = torch.full_like(inp, 0x7f)
        ctx.apply(tmw.D, tmw.ODD, tmw.F32, inp, out)
        got = unpack_multi(ctx, tmw, out, 1, 1, tmw.F32, 4, 4)[0]
        ref = mask_parity(oracle.apply(U, mask_parity(psi, 0), 0.1), 1)
        assert H.per_site_rel_err(got, ref)[0] <= TOL32
