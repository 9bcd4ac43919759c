"""The GCR(k) driver (tmw_options.solver = TMW_GCR; the paper's GPU solver) against the
oracle. The solution of D x = b is unique, so the expected value is the oracle's (BiCGStab, tol 1e-12) solution and the
oracle-recomputed residual; iteration histories are never compared (reading C11)."""
import numpy as np
import pytest

import oracle
from paper_2201_09004_b200 import synth
from test_gpu_parity import SOLVE_CASES, check_solution, dev, make_source

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()
    return m


@pytest.mark.parametrize("precision,nkrylov", [("mixed", 0), ("mixed", 4), ("double", 8)])
@pytest.mark.parametrize("case", SOLVE_CASES)
def test_gcr_solve_vs_oracle(tmw, case, precision, nkrylov):
    L, T, m, c_sw = case["L"], case["T"], case["m"], case["c_sw"]
    scalar = case.get("scalar", False)
    U = synth.gauge_field(L, T, case["eps"], seed=1)
    b = make_source(case)
    x_ref, info_ref = oracle.bicgstab(U, b, m, c_sw, tol=1e-12, mass_reading=int(scalar))
    assert info_ref["status"] == 0
    with tmw.Context(L, T, dev(U), m, c_sw, precision=tmw.MIXED if precision == "mixed" else tmw.DOUBLE, solver=tmw.GCR,
                     nkrylov=nkrylov, mass_reading=tmw.MASS_SCALAR if scalar else tmw.TWIST_GAMMA5) as ctx:
        x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        info = ctx.solve(dev(b), x, 1e-10)
        assert info["true_resid"] <= 1e-10 and info["iters"] > 0 and info["reliable_updates"] >= 1
        check_solution(U, b, x.cpu().numpy(), m, c_sw, x_ref, mass_scalar=scalar)


@pytest.mark.parametrize("precision,nkrylov,c_sw", [("mixed", 4, 1.0509), ("mixed", 0, 0.0), ("double", 3, 1.0509)])
def test_gcr_columns_in_lockstep_vs_oracle(tmw, precision, nkrylov, c_sw):
    """tmw_solve_multi with TMW_GCR steps all columns together (one multi-column Schur application per step); columns of
    different kind leave the steps of a cycle, and the solve, at different times: every column against the oracle."""
    L, T, m = 8, 4, -0.0695 + 0.0j
    U = synth.gauge_field(L, T, 0.4, seed=1)
    F = oracle.field_strength(U) if c_sw else None
    g = synth.gaussian_spinor(L, T, 3)
    b = np.stack([synth.point_source(L, T, 0, 0), synth.z2_source(L, T, 2), g, 1e-4 * g, synth.point_source(L, T, 2, 1),
                  np.zeros_like(g), synth.gaussian_spinor(L, T, 5)])
    n = b.shape[0]
    with tmw.Context(L, T, dev(U), m, c_sw, precision=tmw.MIXED if precision == "mixed" else tmw.DOUBLE, solver=tmw.GCR, nkrylov=nkrylov) as ctx:
        x = torch.empty(b.shape, dtype=torch.complex128, device="cuda")
        k0 = ctx.kernel_counts()
        infos = ctx.solve_multi(n, dev(b), x, 1e-10)
        k1 = ctx.kernel_counts()
        x = x.cpu().numpy()
        assert infos[5]["iters"] == 0 and np.count_nonzero(x[5]) == 0
        steps = 0
        for c in range(n):
            if c == 5:
                continue
            assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0 and infos[c]["reliable_updates"] >= 1
            steps += infos[c]["iters"]
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)
        if precision == "mixed":  # one K1 column application per step and column, issued by multi-column launches
            assert k1["k1_32"] - k0["k1_32"] == steps


def test_gcr_columns_host_and_edge_cases(tmw):
    L, T, m, c_sw = 4, 6, -0.0514 + 0.0j, 1.0424
    U = synth.gauge_field(L, T, 0.35, seed=1)
    F = oracle.field_strength(U)
    b = np.stack([synth.point_source(L, T, 0, 0), np.zeros((T, L, L, L, 4, 3), dtype=np.complex128),
                  synth.point_source(L, T, 3, 2), synth.gaussian_spinor(L, T, 3)])
    with tmw.Context(L, T, U, m, c_sw, location=tmw.HOST, solver=tmw.GCR) as ctx:
        x = np.full(b.shape, 7.0 + 0j)
        infos = ctx.solve_multi(4, b, x, 1e-10)
        assert infos[1]["iters"] == 0 and np.count_nonzero(x[1]) == 0
        for c in (0, 2, 3):
            assert infos[c]["true_resid"] <= 1e-10
            x_ref, _ = oracle.bicgstab(U, b[c], m, c_sw, tol=1e-12, F=F)
            check_solution(U, b[c], x[c], m, c_sw, x_ref, F=F)
    with tmw.Context(L, T, dev(U), m, c_sw, solver=tmw.GCR, max_iter=3) as ctx:
        xg = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        info = ctx.solve(dev(b[3]), xg, 1e-10, allow_noconv=True)
        assert info["status"] == tmw.ENOCONV and info["iters"] == 3 and 1e-10 < info["true_resid"] < 1.0
        r = b[3] - oracle.apply(U, xg.cpu().numpy(), m, c_sw, F=F)
        assert abs(np.linalg.norm(r.ravel()) / np.linalg.norm(b[3].ravel()) - info["true_resid"]) < 1e-9
    for bad in (dict(solver=2), dict(solver=tmw.GCR, nkrylov=17), dict(nkrylov=-1)):
        with pytest.raises(tmw.TmwError) as e:
            tmw.Context(L, T, dev(U), m, c_sw, **bad)
        assert e.value.code == tmw.EINVAL
