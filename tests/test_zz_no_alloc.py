"""tmw_apply_schur_static against tmw_apply_schur (the existing path) on the same packed inputs.

tmw_apply_schur_static is the Schur operator for callers that must not allocate device memory once they are running:
a process whose pooling allocator owns the rest of the card (a raw cudaMalloc then fails or fragments the pool), a job
under a device-memory quota, a loop that cannot take the device-wide stall of cudaMalloc / cudaFree. Its even-parity
intermediate lives in an 8 MiB array compiled into libtmw.so (TMW_STATIC_SCRATCH_BYTES) that every call on the device
shares and that keeps the previous call's contents. So the cases here always make TWO calls in a row, the second on a
different input (and in the other precision, so that the same bytes are reinterpreted): anything stale that leaked from
the first call into the second would show.

Tolerances are the ones of tests/test_gpu_parity.py: per-site relative error <= 1e-5 (fp32), <= 1e-12 (fp64).

This file is named so that pytest collects it LAST: under `pytest -x` a failure here must not hide another test. It
creates its own contexts and depends on nothing another test did, so it passes alone in a fresh process (where its
first call is the one that looks the array's device address up) as well as after the rest of the suite.
"""
import numpy as np
import pytest

import helpers as H
from paper_2201_09004_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {0: 1e-5, 1: 1e-12}  # tmw.F32, tmw.F64


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()  # raises if libtmw.so is missing: no fallback
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def packed(ctx, tmw, psi, prec):
    out = torch.empty(ctx.spinor_bytes(prec), dtype=torch.uint8, device="cuda")
    ctx.pack(prec, tmw.ODD, dev(psi), out)
    return out


def canonical(ctx, tmw, buf, prec, L, T):
    out = torch.zeros((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
    ctx.unpack(prec, tmw.ODD, buf, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("case", [
    dict(L=8, T=16, eps=0.3, m=-0.0695 + 0.01j, c_sw=0.0),   # twisted mass, 2 CTAs-worth of tiles and more
    dict(L=6, T=10, eps=0.4, m=-0.044 + 0.2j, c_sw=1.0349),  # twisted clover, ragged last site block (Vh = 1080)
])
def test_static_scratch_matches_existing_path_twice_in_a_row(tmw, case):
    L, T = case["L"], case["T"]
    U = synth.gauge_field(L, T, case["eps"], seed=5)
    psis = [synth.gaussian_spinor(L, T, seed=11), synth.z2_source(L, T, seed=12)]
    with tmw.Context(L, T, dev(U), case["m"], case["c_sw"]) as ctx:
        # calls in a row on ONE stream (the context's): fp32 D, fp64 D^dag, fp32 D^dag, fp64 D; no clearing in between
        plan = [(tmw.D, tmw.F32, 0), (tmw.DDAG, tmw.F64, 1), (tmw.DDAG, tmw.F32, 1), (tmw.D, tmw.F64, 0)]
        ins = [packed(ctx, tmw, psis[k], prec) for (_, prec, k) in plan]
        outs_new = [torch.full_like(b, 0x7f) for b in ins]
        outs_old = [torch.full_like(b, 0x7f) for b in ins]
        for (op, prec, _), src, dst in zip(plan, ins, outs_new):
            ctx.apply_schur_static(op, prec, src, dst)
        torch.cuda.synchronize()
        for (op, prec, _), src, dst in zip(plan, ins, outs_old):
            ctx.apply_schur(op, prec, src, dst)
        torch.cuda.synchronize()
        for (op, prec, _), new, old in zip(plan, outs_new, outs_old):
            got = canonical(ctx, tmw, new, prec, L, T)
            ref = canonical(ctx, tmw, old, prec, L, T)
            assert np.all(np.isfinite(got)) and np.linalg.norm(ref) > 0
            site, glob = H.per_site_rel_err(got, ref)
            assert site <= TOL[prec], (op, prec, site, glob)
        # and once more after the existing path has run: same answer as the first time
        again = torch.full_like(ins[0], 0x7f)
        ctx.apply_schur_static(plan[0][0], plan[0][1], ins[0], again)
        torch.cuda.synchronize()
        site, _ = H.per_site_rel_err(canonical(ctx, tmw, again, plan[0][1], L, T), canonical(ctx, tmw, outs_old[0], plan[0][1], L, T))
        assert site <= TOL[plan[0][1]], site


def test_static_scratch_refuses_what_does_not_fit(tmw):
    """16^3 x 32: the fp32 parity spinor (6 MiB) fits the 8 MiB array, the fp64 one (12 MiB) does not -> TMW_EINVAL with
    both sizes in the text, and nothing is launched. Decomposed contexts are refused as well."""
    L, T = 16, 32
    U = synth.gauge_field(L, T, 0.3, seed=7)
    psi = synth.gaussian_spinor(L, T, seed=8)
    with tmw.Context(L, T, dev(U), 0.1 + 0.0j, 0.0) as ctx:
        assert ctx.spinor_bytes(tmw.F32) <= tmw.STATIC_SCRATCH_BYTES < ctx.spinor_bytes(tmw.F64)
        src = packed(ctx, tmw, psi, tmw.F32)
        dst = torch.empty_like(src)
        ref = torch.empty_like(src)
        ctx.apply_schur_static(tmw.D, tmw.F32, src, dst)
        ctx.apply_schur(tmw.D, tmw.F32, src, ref)
        site, _ = H.per_site_rel_err(canonical(ctx, tmw, dst, tmw.F32, L, T), canonical(ctx, tmw, ref, tmw.F32, L, T))
        assert site <= TOL[tmw.F32], site
        src64 = packed(ctx, tmw, psi, tmw.F64)
        dst64 = torch.full_like(src64, 0x5a)
        n0 = ctx.launch_count()
        with pytest.raises(tmw.TmwError) as ei:
            ctx.apply_schur_static(tmw.D, tmw.F64, src64, dst64)
        assert ei.value.code == tmw.EINVAL
        assert str(ctx.spinor_bytes(tmw.F64)) in str(ei.value) and str(tmw.STATIC_SCRATCH_BYTES) in str(ei.value)
        assert ctx.launch_count() == n0
        torch.cuda.synchronize()
        assert bool((dst64 == 0x5a).all())
    Ls, Ts = 4, 8
    with tmw.Context(Ls, Ts, dev(synth.gauge_field(Ls, Ts, 0.3, seed=1)), 0.1 + 0.0j, 0.0, domains_t=2) as ctx:
        buf = torch.zeros(ctx.spinor_bytes(tmw.F32), dtype=torch.uint8, device="cuda")
        with pytest.raises(tmw.TmwError) as ei:
            ctx.apply_schur_static(tmw.D, tmw.F32, buf, torch.empty_like(buf))
        assert ei.value.code == tmw.EINVAL
