"""Parity of the fused gamma5 D (TMW_G5D) and of the Clenshaw-evaluated Chebyshev series of gamma5 D
(tmw_cheb_apply) with the fp64 oracle. Tolerances as in test_gpu_parity.py; the series
adds up ncoef applications, so its fp64 tolerance is 1e-12 relative to the largest site norm of the result."""
import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth
from test_gpu_parity import TOL32, TOL64, dev, gpu_pack, gpu_unpack, mask_parity, packed_empty

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()
    return m


CASES = [dict(L=4, T=8, eps=0.3, m=-1.5 + 0.0j, c_sw=0.0),      # the overlap kernel D_w(-rho), rho = 1.5
         dict(L=6, T=4, eps=0.4, m=-0.0695 + 0.0j, c_sw=1.0509),
         dict(L=4, T=6, eps=0.3, m=-0.044 + 0.2j, c_sw=1.0349)]


@pytest.mark.parametrize("case", CASES)
def test_gamma5_D_full_and_parity_vs_oracle(tmw, case):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[:, None]
    with tmw.Context(L, T, dev(U), m, c_sw) as ctx:
        out = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        ctx.apply(tmw.G5D, tmw.FULL, tmw.F64, dev(psi), out)
        torch.cuda.synchronize()
        site, glob = H.per_site_rel_err(out.cpu().numpy(), oracle.gamma5_apply(U, psi, m, c_sw))
        assert site <= TOL64, (site, glob)
        for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
            for par in (0, 1):
                inp = gpu_pack(ctx, tmw, psi, 1 - par, prec)
                o = packed_empty(ctx, tmw, prec)
                ctx.apply(tmw.G5D, tmw.ODD if par else tmw.EVEN, prec, inp, o)
                got = gpu_unpack(ctx, tmw, o, par, prec, L, T)
                # on parity p only the hopping term of D acts on a source living on parity pbar; then gamma5
                ref = g5 * mask_parity(oracle.apply(U, mask_parity(psi, 1 - par), m, c_sw), par)
                site, glob = H.per_site_rel_err(got, ref)
                assert site <= tol, (prec, par, site, glob)


@pytest.mark.parametrize("case", CASES[:2])
@pytest.mark.parametrize("ncoef", [1, 2, 3, 16])
def test_cheb_apply_vs_oracle(tmw, case, ncoef):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    coef = np.random.default_rng(7).standard_normal(ncoef)
    scale, shift = 0.12, 0.03  # |gamma5 D| <= 8 + |m| on any field: the spectrum of X stays inside [-1, 1]
    ref = oracle.cheb_series(U, psi, coef, scale, shift, m, c_sw)
    tol = TOL64 * max(1, ncoef)
    with tmw.Context(L, T, dev(U), m, c_sw) as ctx:
        out = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        ctx.cheb_apply(coef, scale, shift, dev(psi), out)
        torch.cuda.synchronize()
        err = np.linalg.norm((out.cpu().numpy() - ref).reshape(-1, 12), axis=1).max() / np.linalg.norm(ref.reshape(-1, 12), axis=1).max()
        assert err <= tol, err
    with tmw.Context(L, T, U, m, c_sw, location=tmw.HOST) as ctx:
        o = np.empty_like(psi)
        ctx.cheb_apply(coef, scale, shift, psi, o)
        err = np.linalg.norm((o - ref).reshape(-1, 12), axis=1).max() / np.linalg.norm(ref.reshape(-1, 12), axis=1).max()
        assert err <= tol, err


def test_cheb_apply_errors(tmw):
    U = dev(synth.gauge_field(4, 4, 0.3, seed=1))
    with tmw.Context(4, 4, U, 0.1) as ctx:
        x = torch.zeros((4, 4, 4, 4, 4, 3), dtype=torch.complex128, device="cuda")
        y = torch.empty_like(x)
        for bad in (dict(coef=[], src=x, dst=y), dict(coef=[1.0, float("nan")], src=x, dst=y), dict(coef=[1.0], src=x, dst=x)):
            with pytest.raises(tmw.TmwError) as e:
                ctx.cheb_apply(bad["coef"], 1.0, 0.0, bad["src"], bad["dst"])
            assert e.value.code == tmw.EINVAL
