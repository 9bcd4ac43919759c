"""Parity of the persistent link-ring fp32 stencil (csrc/tmw_dslash_ring.cuh, tmw_options.ring = 1: CTAs walk over the site
blocks, every thread prefetches the 8 links of its next site into private shared-memory slots with cp.async) with the fp64
CPU oracle, on identical seeded inputs: hop, K1 / K2 with every kind of diagonal part, 1-4 columns per thread (packed
pairs for even counts), lattices whose site count is not a multiple of the CTA size (idle lanes in the last block),
fewer site blocks than resident CTAs and many more, the fused dot products through a 12-column solve."""
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


def ring_launches(ctx, fn):
    before = ctx.kernel_counts()
    fn()
    after = ctx.kernel_counts()
    n = after["ring"] - before["ring"]
    assert n == sum(after[k] - before[k] for k in ("hop32", "k1_32", "k2_32", "k2_32_dots"))
    return n


@pytest.mark.parametrize("L,T,nrhs,cpt,zchunk", [(8, 4, 5, 2, 0), (8, 4, 3, 3, 4), (6, 4, 7, 4, 0), (6, 4, 1, 0, 0), (4, 8, 6, 1, 0),
                                                  (16, 32, 2, 2, 0), (16, 32, 1, 0, 0)])
def test_hopping_ring_vs_oracle(tmw, L, T, nrhs, cpt, zchunk):
    U = synth.gauge_field(L, T, 0.4, seed=1)
    cols = columns(L, T, nrhs)
    with tmw.Context(L, T, dev(U), 0.1, ring=1, columns_per_thread=cpt, zchunk=zchunk) as ctx:
        for op in (tmw.D, tmw.DDAG, tmw.G5D):
            for par in (0, 1):
                inp = pack_multi(ctx, tmw, cols, 1 - par, tmw.F32)
                out = torch.full_like(inp, 0x7f)
                assert ring_launches(ctx, lambda: ctx.apply_multi(op, tmw.ODD if par else tmw.EVEN, tmw.F32, nrhs, inp, out)) == nrhs
                got = unpack_multi(ctx, tmw, out, nrhs, par, tmw.F32, L, T)
                for c in range(nrhs):
                    if L == 16 and c > 0:
                        continue  # one column of the large lattice against the oracle is enough
                    ref = mask_parity(oracle.apply(U, mask_parity(cols[c], 1 - par), 0.1, dagger=(op == tmw.DDAG)), par)
                    if op == tmw.G5D:
                        ref = ref * np.array([1, 1, -1, -1])[:, None]
                    site, glob = H.per_site_rel_err(got[c], ref)
                    assert site <= TOL32, (op, par, c, site, glob)


@pytest.mark.parametrize("cpt", [1, 2, 3, 4])
@pytest.mark.parametrize("case", [
    dict(L=8, T=4, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509, nrhs=5),
    dict(L=4, T=6, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349, nrhs=4),   # twisted clover: two-factor inverse
    dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.01j, c_sw=0.0, nrhs=6),    # twisted mass, no clover
])
def test_schur_ring_vs_oracle(tmw, case, cpt):
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
    with tmw.Context(L, T, dev(U), m, c_sw, ring=1, columns_per_thread=cpt) as ctx:
        inp = pack_multi(ctx, tmw, cols, 1, tmw.F32)
        out = torch.full_like(inp, 0x7f)
        assert ring_launches(ctx, lambda: ctx.apply_schur_multi(tmw.D, tmw.F32, nrhs, inp, out)) == 2 * nrhs
        got = unpack_multi(ctx, tmw, out, nrhs, 1, tmw.F32, L, T)
        for c in range(nrhs):
            site, glob = H.per_site_rel_err(got[c], refs[c])
            assert site <= TOL32, (c, site, glob)


@pytest.mark.parametrize("c_sw,m", [(1.0424, -0.0514 + 0.0j), (0.0, -0.0695 + 0.01j)])
def test_solve_multi_ring_vs_oracle(tmw, c_sw, m):
    L, T = 8, 4
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U) if c_sw else None
    b = np.stack([synth.point_source(L, T, c // 3, c % 3) for c in range(12)])
    with tmw.Context(L, T, dev(U), m, c_sw, ring=1) as ctx:
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        infos = ctx.solve_multi(12, dev(b), x, 1e-10)
        assert ctx.kernel_counts()["ring"] > 0
        x = x.cpu().numpy()
        for c in range(12):
            assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)


def test_ring_falls_back(tmw):
    """18-real links and bad option values: the plain kernel / TMW_EINVAL"""
    U = synth.gauge_field(4, 4, 0.3, seed=1)
    for kw in (dict(ring=2), dict(ring=-2)):
        with pytest.raises(tmw.TmwError) as e:
            tmw.Context(4, 4, dev(U), 0.1, **kw)
        assert e.value.code == tmw.EINVAL
    psi = synth.gaussian_spinor(4, 4, seed=3)
    with tmw.Context(4, 4, dev(U), 0.1, ring=1, reconstruct=18) as ctx:
        inp = pack_multi(ctx, tmw, [psi], 0, tmw.F32)
        out = torch.full_like(inp, 0x7f)
        ctx.apply(tmw.D, tmw.ODD, tmw.F32, inp, out)
        assert ctx.kernel_counts()["ring"] == 0
        got = unpack_multi(ctx, tmw, out, 1, 1, tmw.F32, 4, 4)[0]
        ref = mask_parity(oracle.apply(U, mask_parity(psi, 0), 0.1), 1)
        assert H.per_site_rel_err(got, ref)[0] <= TOL32
