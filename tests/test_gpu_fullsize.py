"""Parity at BASELINE.json's full sizes (configs[1..4]) in the launch configuration bench.py times (fp32 12-real gauge,
packed parity spinors, tmw_apply EVEN|ODD / tmw_apply FULL / tmw_solve through the C ABI).

The oracle cannot sweep these lattices many times in seconds, so:
  * operator outputs are compared with the oracle ONE SITE AT A TIME (oracle.apply_sites) on a seeded sample of
    sites plus every kind of boundary site (x, y, z wrap; the antiperiodic t wrap) — tolerance as in
    test_gpu_parity.py (fp32 1e-5, fp64 1e-12 per site);
  * solutions: the EXACT full-lattice residual |b - D x| / |b| <= 1e-10 with D applied by the oracle over the whole
    lattice (oracle.apply with its precomputed F; seconds at these sizes), on every config; and
    |x_gpu - x_oracle| / |x_oracle| <= 1e-8 against the oracle's own solution (oracle.bicgstab to 1e-12): over the whole
    lattice on configs 1-3, and on config 4 against the sample of the oracle's solution stored in
    tests/golden/cfg4_solution_sample.txt (written by tests/golden/make_cfg4_solution_sample.py, which imports only
    oracle/ and the input generators; the solve takes ~48 GB of host memory and tens of minutes).
"""
import os
import numpy as np
import pytest

import helpers as H
import oracle
from paper_2201_09004_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL32, TOL64 = 1e-5, 1e-12
_cache = {}


@pytest.fixture(scope="module")
def tmw():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_09004_b200 import tmw as m
    m.load()
    return m


def config_fields(idx):
    """(cfg, U) of BASELINE.json configs[idx]; one field is kept at a time (the largest is 9.2 GB)."""
    if _cache.get("idx") != idx:
        _cache.clear()
        cfg = synth.CONFIGS[idx]
        _cache.update(idx=idx, cfg=cfg, U=synth.gauge_field(cfg["L"], cfg["T"], cfg["eps"], seed=1))
    return _cache["cfg"], _cache["U"]


def config_F(idx):
    """the oracle's clover-leaf field strength of configs[idx] (13.8 GB at 48^3 x 144), cached with the gauge field"""
    cfg, U = config_fields(idx)
    if cfg["c_sw"] == 0:
        return None
    if "F" not in _cache:
        _cache["F"] = oracle.field_strength(U)
    return _cache["F"]


def exact_residual(U, F, b, x, m, c_sw):
    """|b - D x| / |b| over the WHOLE lattice, D applied by the oracle (Eq. (2) + :67 Eq. (3))"""
    r = b - oracle.apply(U, x, m, c_sw, F=F)
    return float(np.linalg.norm(r.ravel()) / np.linalg.norm(b.ravel()))


def lex(L, x, y, z, t):
    return x + L * (y + L * (z + L * t))


def random_sites(L, T, n, seed):
    return np.unique(np.random.default_rng(seed).integers(0, L ** 3 * T, size=n)).astype(np.int64)


def boundary_sites(L, T):
    edge = [0, 1, L - 2, L - 1]
    tedge = [0, 1, T - 2, T - 1]
    return np.unique(np.array([lex(L, x, y, z, t) for t in tedge for z in edge for y in edge for x in edge], dtype=np.int64))


def sample_sites(L, T, n, seed, parity=None):
    """n seeded random sites + boundary sites of every kind (lexicographic indices), optionally of one parity."""
    rng = np.random.default_rng(seed)
    V = L ** 3 * T
    s = list(rng.integers(0, V, size=n))
    edge = [0, 1, L - 2, L - 1]
    tedge = [0, 1, T - 2, T - 1]
    for t in tedge:
        for z in edge:
            for y in edge:
                for x in edge:
                    s.append(lex(L, x, y, z, t))
    s = np.unique(np.array(s, dtype=np.int64))
    if parity is not None:
        x = s % L
        y = (s // L) % L
        z = (s // (L * L)) % L
        t = s // (L ** 3)
        s = s[(x + y + z + t) % 2 == parity]
    return s


def mask_parity_inplace(psi, L, T, par_zero):
    flat = psi.reshape(-1, 12)
    flat[H.parity_sites(L, T, par_zero)] = 0
    return psi


def site_err(got, ref):
    rn = np.linalg.norm(ref.reshape(-1, 12), axis=1)
    dn = np.linalg.norm((got - ref).reshape(-1, 12), axis=1)
    assert np.all(rn > 0)
    return float(np.max(dn / rn))


@pytest.mark.parametrize("idx", [1, 3, 4])
def test_fullsize_hopping_fp32_sampled(tmw, idx):
    cfg, U = config_fields(idx)
    L, T, m = cfg["L"], cfg["T"], complex(*cfg["m"])
    psi = synth.gaussian_spinor(L, T, seed=3)
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, cfg["c_sw"]) as ctx:
        del dU
        dpsi = torch.from_numpy(psi).cuda()
        out_c = torch.zeros_like(dpsi)
        nb = ctx.spinor_bytes(tmw.F32)
        pin = torch.empty(nb, dtype=torch.uint8, device="cuda")
        pout = torch.empty(nb, dtype=torch.uint8, device="cuda")
        for op in (tmw.D, tmw.DDAG):
            for par in (0, 1):
                ctx.pack(tmw.F32, tmw.EVEN if par else tmw.ODD, dpsi, pin)  # input lives on parity 1 - par
                ctx.apply(op, tmw.ODD if par else tmw.EVEN, tmw.F32, pin, pout)
                ctx.unpack(tmw.F32, tmw.ODD if par else tmw.EVEN, pout, out_c)
            torch.cuda.synchronize()
            got_full = out_c.cpu().numpy().reshape(-1, 4, 3)
            # the oracle's full D on psi gives hop + A psi(x); the hopping block alone is D with the site term
            # removed: apply_sites with c_sw = 0 and subtract the mass term -(4+m) psi (twist is 0 or handled below)
            sites = sample_sites(L, T, 20000, seed=11 + idx)
            ref = oracle.apply_sites(U, psi, sites, m, 0.0, dagger=(op == tmw.DDAG))
            p = psi.reshape(-1, 4, 3)[sites]
            tw = -m.imag if op == tmw.D else m.imag
            g5 = np.array([1, 1, -1, -1])[None, :, None]
            ref = ref - (-(4.0 + m.real) * p + 1j * tw * g5 * p)
            assert site_err(got_full[sites], ref) <= TOL32
        del dpsi, out_c, pin, pout
    torch.cuda.empty_cache()


@pytest.mark.parametrize("idx,ncol", [(3, 12), (4, 3)])
def test_fullsize_hopping_multi_column_fp32_sampled(tmw, idx, ncol):
    """the multi-column hop launches of bench.py's `multi_rhs` leg (tmw_apply_multi; automatic columns per thread, packed
    fp32 pairs, z-slab sweep, link prefetch): every column at sampled sites incl. all boundary kinds against the oracle"""
    cfg, U = config_fields(idx)
    L, T, m = cfg["L"], cfg["T"], complex(*cfg["m"])
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, cfg["c_sw"]) as ctx:
        del dU
        nb = ctx.spinor_bytes(tmw.F32)
        pin = torch.empty(nb * ncol, dtype=torch.uint8, device="cuda")
        pout = torch.full_like(pin, 0x7f)
        tmp = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        seeds = [20 + c for c in range(ncol)]
        for c in range(ncol):
            tmp.copy_(torch.from_numpy(synth.gaussian_spinor(L, T, seed=seeds[c])))
            ctx.pack(tmw.F32, tmw.EVEN, tmp, pin[c * nb:(c + 1) * nb])
        ctx.apply_multi(tmw.D, tmw.ODD, tmw.F32, ncol, pin, pout)
        sites = sample_sites(L, T, 4000, seed=31 + idx, parity=1)
        for c in range(ncol):
            tmp.zero_()
            ctx.unpack(tmw.F32, tmw.ODD, pout[c * nb:(c + 1) * nb], tmp)
            got = tmp.cpu().numpy().reshape(-1, 4, 3)[sites]
            psi = synth.gaussian_spinor(L, T, seed=seeds[c])
            mask_parity_inplace(psi, L, T, 1)  # the input lives on the even sites
            ref = oracle.apply_sites(U, psi, sites, m, 0.0)  # at odd sites of an even-only input: the hopping block alone
            assert site_err(got, ref) <= TOL32, c
        del pin, pout, tmp
    torch.cuda.empty_cache()


@pytest.mark.parametrize("idx", [2, 4])
def test_fullsize_full_operator_fp64_sampled(tmw, idx):
    cfg, U = config_fields(idx)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    psi = synth.gaussian_spinor(L, T, seed=3)
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        dpsi = torch.from_numpy(psi).cuda()
        out = torch.empty_like(dpsi)
        sites = sample_sites(L, T, 5000, seed=21 + idx)
        for op in (tmw.D, tmw.DDAG):
            ctx.apply(op, tmw.FULL, tmw.F64, dpsi, out)
            torch.cuda.synchronize()
            got = out.cpu().numpy().reshape(-1, 4, 3)[sites]
            ref = oracle.apply_sites(U, psi, sites, m, c_sw, dagger=(op == tmw.DDAG))
            assert site_err(got, ref) <= TOL64
        del dpsi, out
    torch.cuda.empty_cache()


@pytest.mark.parametrize("idx", [1, 2])
def test_fullsize_solve_vs_oracle_solution(tmw, idx):
    cfg, U = config_fields(idx)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    b = synth.z2_source(L, T, 2) if cfg["source"] == "z2" else synth.point_source(L, T, 0, 0)
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        info = ctx.solve(torch.from_numpy(b).cuda(), x, 1e-10)
        xg = x.cpu().numpy()
        del x
    torch.cuda.empty_cache()
    assert info["true_resid"] <= 1e-10
    F = oracle.field_strength(U) if c_sw != 0 else None
    r = b - oracle.apply(U, xg, m, c_sw, F=F)
    assert np.linalg.norm(r.ravel()) / np.linalg.norm(b.ravel()) <= 1e-10
    x_ref, iref = oracle.bicgstab(U, b, m, c_sw, tol=1e-12, F=F)
    assert iref["status"] == 0
    assert np.linalg.norm((xg - x_ref).ravel()) / np.linalg.norm(x_ref.ravel()) <= 1e-8


def test_fullsize_schur_fp32_sampled(tmw):
    """The fp32 clover K1/K2 kernels (A4/A5) at full size in the launch configuration of the solver: tmw_apply_schur on
    configs[2] (24^3 x 64, c_sw = 1.0509) against the oracle's masked pieces, Mhat p_o = A_oo p_o - H_oe A_ee^{-1} H_eo p_o
    with A_ee^{-1} by a dense 12 x 12 solve per site (numpy) of the oracle's site term; compared per site on ALL odd
    sites (fp32 <= 1e-5, fp64 <= 1e-12)."""
    idx = 2
    cfg, U = config_fields(idx)
    F = config_F(idx)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    V = L ** 3 * T
    psi = synth.gaussian_spinor(L, T, seed=3)
    ev, od = H.parity_sites(L, T, 0), H.parity_sites(L, T, 1)
    blocks = H.site_diagonal_blocks(U, c_sw, m.real)[ev]          # (Vh, 2, 6, 6) Hermitian chirality blocks on even sites
    x_o = mask_parity_inplace(psi.copy(), L, T, 0)
    Dx = oracle.apply(U, x_o, m, c_sw, F=F).reshape(V, 12)       # even: H_eo x_o; odd: A_oo x_o
    t_e = np.zeros((V, 12), dtype=np.complex128)
    rhs = Dx[ev].reshape(-1, 2, 6, 1)
    t_e[ev] = np.linalg.solve(blocks, rhs).reshape(-1, 12)
    Dt = oracle.apply(U, t_e.reshape(psi.shape), m, c_sw, F=F).reshape(V, 12)  # odd: H_oe t_e (+ A_oo 0)
    ref = np.zeros((V, 12), dtype=np.complex128)
    ref[od] = Dx[od] - Dt[od]
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        dpsi = torch.from_numpy(psi).cuda()
        for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
            nb = ctx.spinor_bytes(prec)
            pin = torch.empty(nb, dtype=torch.uint8, device="cuda")
            pout = torch.empty(nb, dtype=torch.uint8, device="cuda")
            out_c = torch.zeros_like(dpsi)
            ctx.pack(prec, tmw.ODD, dpsi, pin)
            ctx.apply_schur(tmw.D, prec, pin, pout)
            ctx.unpack(prec, tmw.ODD, pout, out_c)
            torch.cuda.synchronize()
            got = out_c.cpu().numpy().reshape(V, 12)
            assert site_err(got[od], ref[od]) <= tol, prec
        del dpsi, out_c, pin, pout
    torch.cuda.empty_cache()


def neighbours(L, T, sites):
    """the 8 nearest neighbours (periodic index arithmetic; the antiperiodic sign is the operator's business) of each site"""
    x, y, z, t = sites % L, (sites // L) % L, (sites // (L * L)) % L, sites // (L ** 3)
    out = []
    for d in (1, -1):
        out += [lex(L, (x + d) % L, y, z, t), lex(L, x, (y + d) % L, z, t), lex(L, x, y, (z + d) % L, t), lex(L, x, y, z, (t + d) % T)]
    return np.unique(np.concatenate(out)).astype(np.int64)


class SchurSampledRef:
    """Mhat p_o = A_oo p_o - H_oe A_ee^{-1} H_eo p_o at a list S of odd sites, from the oracle's per-site routine only
    (oracle.apply_sites; no full-lattice sweep, so it works at 48^3 x 144): with N = the even neighbours of S,
      h_N = (D p_o)(N)  (p_o lives on odd sites, so at an even site this is the hopping block alone),
      A(x) for x in N column by column from D applied to unit vectors placed on N (even sites do not see one another),
      t_N = A^{-1} h_N by a dense 12 x 12 solve per site (numpy), t = 0 elsewhere,
      ref(S) = (D p_o)(S) - (D t)(S)  (at an odd site: A_oo p_o, and the hopping block of the even field t).
    The site matrices depend on the fields only and are shared by all columns."""

    def __init__(self, U, m, c_sw, S, dagger=False):
        self.U, self.m, self.c_sw, self.S, self.dagger = U, m, c_sw, S, dagger
        T, L = U.shape[1], U.shape[2]
        self.L, self.T = L, T
        self.N = neighbours(L, T, S)
        xs = self.N % L + (self.N // L) % L + (self.N // (L * L)) % L + self.N // (L ** 3)
        assert np.all(xs % 2 == 0), "S must hold odd sites only"
        self.work = np.zeros((T, L, L, L, 4, 3), dtype=np.complex128)
        flat = self.work.reshape(-1, 12)
        A = np.empty((self.N.size, 12, 12), dtype=np.complex128)
        for k in range(12):
            flat[self.N, k] = 1.0
            A[:, :, k] = oracle.apply_sites(U, self.work, self.N, m, c_sw, dagger=dagger).reshape(-1, 12)
            flat[self.N, k] = 0.0
        self.A = A

    def __call__(self, p_o):
        """p_o: canonical spinor that vanishes on the even sites -> (len(S), 4, 3)"""
        h = oracle.apply_sites(self.U, p_o, self.N, self.m, self.c_sw, dagger=self.dagger).reshape(-1, 12)
        flat = self.work.reshape(-1, 12)
        flat[self.N] = np.linalg.solve(self.A, h[..., None])[..., 0]
        ref = oracle.apply_sites(self.U, p_o, self.S, self.m, self.c_sw, dagger=self.dagger) - \
            oracle.apply_sites(self.U, self.work, self.S, self.m, self.c_sw, dagger=self.dagger)
        flat[self.N] = 0.0
        return ref


def test_schur_sampled_reference_agrees_with_the_full_lattice_one():
    """the sampled reference above against the whole-lattice construction of test_fullsize_schur_fp32_sampled on a small
    lattice (both from the oracle; this checks the test's own bookkeeping, not the product)"""
    L, T, m, c_sw = 4, 6, -0.044 + 0.2j, 1.0349
    U = synth.gauge_field(L, T, 0.4, seed=1)
    V = L ** 3 * T
    psi = mask_parity_inplace(synth.gaussian_spinor(L, T, seed=3), L, T, 0)
    ev, od = H.parity_sites(L, T, 0), H.parity_sites(L, T, 1)
    Dx = oracle.apply(U, psi, m, c_sw).reshape(V, 12)
    A = np.empty((V, 12, 12), dtype=np.complex128)
    e = np.zeros((V, 12), dtype=np.complex128)
    for k in range(12):
        e[ev, k] = 1.0
        A[:, :, k] = oracle.apply(U, e.reshape(psi.shape), m, c_sw).reshape(V, 12)
        e[ev, k] = 0.0
    t_e = np.zeros((V, 12), dtype=np.complex128)
    t_e[ev] = np.linalg.solve(A[ev], Dx[ev][..., None])[..., 0]
    ref = Dx - oracle.apply(U, t_e.reshape(psi.shape), m, c_sw).reshape(V, 12)
    S = od[::7]
    got = SchurSampledRef(U, m, c_sw, S)(psi).reshape(-1, 12)
    assert np.max(np.abs(got - ref[S])) <= 1e-13 * np.max(np.abs(ref))


@pytest.mark.parametrize("idx,ncol", [(3, 12), (4, 3)])
def test_fullsize_schur_single_and_multi_column_sampled(tmw, idx, ncol):
    """K1/K2 at the sizes and in the launch shapes bench.py times, against the oracle site by site (not through a converging
    solve): tmw_apply_schur_multi on `ncol` columns (fp32: columns per thread, packed pairs, z-slab sweep) and
    tmw_apply_schur on one column in fp32 and fp64, at 1500 seeded odd sites plus the odd boundary sites of every kind."""
    cfg, U = config_fields(idx)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    S = sample_sites(L, T, 3000, seed=41 + idx, parity=1)
    ref_of = SchurSampledRef(U, m, c_sw, S)
    seeds = [50 + c for c in range(ncol)]
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        tmp = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        nb = ctx.spinor_bytes(tmw.F32)
        pin = torch.empty(nb * ncol, dtype=torch.uint8, device="cuda")
        pout = torch.full_like(pin, 0x7f)
        for c in range(ncol):
            tmp.copy_(torch.from_numpy(synth.gaussian_spinor(L, T, seed=seeds[c])))
            ctx.pack(tmw.F32, tmw.ODD, tmp, pin[c * nb:(c + 1) * nb])
        ctx.apply_schur_multi(tmw.D, tmw.F32, ncol, pin, pout)
        for c in range(ncol):
            tmp.zero_()
            ctx.unpack(tmw.F32, tmw.ODD, pout[c * nb:(c + 1) * nb], tmp)
            got = tmp.cpu().numpy().reshape(-1, 4, 3)[S]
            psi = mask_parity_inplace(synth.gaussian_spinor(L, T, seed=seeds[c]), L, T, 0)
            ref = ref_of(psi)
            assert site_err(got, ref) <= TOL32, ("multi", c)
            if c == 0:  # the single-column launches on the same input, fp32 and fp64
                for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
                    n1 = ctx.spinor_bytes(prec)
                    a = torch.empty(n1, dtype=torch.uint8, device="cuda")
                    o = torch.full_like(a, 0x7f)
                    tmp.copy_(torch.from_numpy(psi))
                    ctx.pack(prec, tmw.ODD, tmp, a)
                    ctx.apply_schur(tmw.D, prec, a, o)
                    tmp.zero_()
                    ctx.unpack(prec, tmw.ODD, o, tmp)
                    assert site_err(tmp.cpu().numpy().reshape(-1, 4, 3)[S], ref) <= tol, ("single", prec)
                    del a, o
        del pin, pout, tmp
    torch.cuda.empty_cache()


def cut_plane_sites(L, T, pz, pt):
    """every site next to a domain cut: z in {0, lz-1, lz, ...} for domains_z > 1, t likewise (lexicographic indices)"""
    zs = sorted({(k * (L // pz) + d) % L for k in range(pz) for d in (-1, 0)}) if pz > 1 else []
    ts = sorted({(k * (T // pt) + d) % T for k in range(pt) for d in (-1, 0)}) if pt > 1 else []
    ax, ay = np.arange(L), np.arange(L)
    out = []
    for z in zs:
        t, y, x = np.meshgrid(np.arange(T), ay, ax, indexing="ij")
        out.append(lex(L, x, y, z, t).ravel())
    for t in ts:
        z, y, x = np.meshgrid(np.arange(L), ay, ax, indexing="ij")
        out.append(lex(L, x, y, z, t).ravel())
    return np.unique(np.concatenate(out)).astype(np.int64)


def of_parity(L, sites, par):
    return sites[((sites % L) + (sites // L) % L + (sites // (L * L)) % L + sites // (L ** 3)) % 2 == par]


@pytest.mark.parametrize("idx,pz,pt", [(3, 2, 2), (4, 1, 2)])
def test_fullsize_decomposed_context_sampled(tmw, idx, pz, pt):
    """Domain-decomposed contexts at full size - 2 x 2 domains at configs[3], the 1 x 2 split bench.py times
    at configs[4] - where the local site mapping, the vh_loc-strided buffers and the face indices span many CTAs: the fp32
    hopping block and the fp64 FULL operator at EVERY site next to a cut plus 5000 seeded sites and the lattice-boundary
    sites; K1/K2 (tmw_apply_schur, fp32 and fp64) at a seeded sample of those; one solve with the exact residual through the
    oracle's D. All against the oracle site by site (oracle.apply_sites)."""
    cfg, U = config_fields(idx)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    cuts = cut_plane_sites(L, T, pz, pt)
    sites = np.unique(np.concatenate([cuts, sample_sites(L, T, 5000, seed=61 + idx)]))
    rng = np.random.default_rng(71 + idx)
    S = np.unique(np.concatenate([rng.choice(of_parity(L, cuts, 1), size=2000, replace=False),
                                  sample_sites(L, T, 2000, seed=81 + idx, parity=1)]))
    psi = synth.gaussian_spinor(L, T, seed=3)
    psi_o = mask_parity_inplace(psi.copy(), L, T, 0)
    ref_schur = SchurSampledRef(U, m, c_sw, S)(psi_o)
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw, domains_z=pz, domains_t=pt) as ctx:
        del dU
        dpsi = torch.from_numpy(psi).cuda()
        out_c = torch.zeros_like(dpsi)
        # fp32 hopping block, both parities
        nb = ctx.spinor_bytes(tmw.F32)
        pin = torch.empty(nb, dtype=torch.uint8, device="cuda")
        pout = torch.full_like(pin, 0x7f)
        for par in (0, 1):
            ctx.pack(tmw.F32, tmw.EVEN if par else tmw.ODD, dpsi, pin)
            ctx.apply(tmw.D, tmw.ODD if par else tmw.EVEN, tmw.F32, pin, pout)
            ctx.unpack(tmw.F32, tmw.ODD if par else tmw.EVEN, pout, out_c)
        torch.cuda.synchronize()
        got = out_c.cpu().numpy().reshape(-1, 4, 3)[sites]
        p = psi.reshape(-1, 4, 3)[sites]
        g5 = np.array([1, 1, -1, -1])[None, :, None]
        ref = oracle.apply_sites(U, psi, sites, m, 0.0) - (-(4.0 + m.real) * p - 1j * m.imag * g5 * p)  # D (c_sw = 0) minus its site term
        assert site_err(got, ref) <= TOL32
        # K1 / K2
        for prec, tol in ((tmw.F32, TOL32), (tmw.F64, TOL64)):
            n1 = ctx.spinor_bytes(prec)
            a = torch.empty(n1, dtype=torch.uint8, device="cuda")
            o = torch.full_like(a, 0x7f)
            ctx.pack(prec, tmw.ODD, dpsi, a)
            ctx.apply_schur(tmw.D, prec, a, o)
            out_c.zero_()
            ctx.unpack(prec, tmw.ODD, o, out_c)
            assert site_err(out_c.cpu().numpy().reshape(-1, 4, 3)[S], ref_schur) <= tol, prec
            del a, o
        del pin, pout
        # fp64 FULL operator
        ctx.apply(tmw.D, tmw.FULL, tmw.F64, dpsi, out_c)
        torch.cuda.synchronize()
        assert site_err(out_c.cpu().numpy().reshape(-1, 4, 3)[sites], oracle.apply_sites(U, psi, sites, m, c_sw)) <= TOL64
        # one solve, residual by the oracle's operator over the whole lattice
        b = synth.point_source(L, T, 0, 0)
        dpsi.copy_(torch.from_numpy(b))
        info = ctx.solve(dpsi, out_c, 1e-10)
        xg = out_c.cpu().numpy()
        del dpsi, out_c
    torch.cuda.empty_cache()
    assert info["true_resid"] <= 1e-10
    assert exact_residual(U, config_F(idx), b, xg, m, c_sw) <= 1e-10


ORIGIN_COLS = [(0, 0), (2, 1)]  # (spin, colour) of the columns whose solution is compared with the oracle's at config 3


def test_fullsize_config3_twelve_columns(tmw):
    """configs[3]: the 12 point sources of a propagator, one after another. Every column: exact
    full-lattice residual through the oracle's D. Columns (0,0) and (2,1): the solution against the oracle's."""
    cfg, U = config_fields(3)
    F = config_F(3)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    dU = torch.from_numpy(U).cuda()
    sols = {}
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        for spin in range(4):
            for colour in range(3):
                b = synth.point_source(L, T, spin, colour)
                info = ctx.solve(torch.from_numpy(b).cuda(), x, 1e-10)
                assert info["true_resid"] <= 1e-10
                xg = x.cpu().numpy()
                assert exact_residual(U, F, b, xg, m, c_sw) <= 1e-10, (spin, colour)
                if (spin, colour) in ORIGIN_COLS:
                    sols[(spin, colour)] = xg
        del x
    torch.cuda.empty_cache()
    for (spin, colour), xg in sols.items():
        x_ref, iref = oracle.bicgstab(U, synth.point_source(L, T, spin, colour), m, c_sw, tol=1e-12, F=F)
        assert iref["status"] == 0 and iref["true_resid"] <= 1e-11
        assert np.linalg.norm((xg - x_ref).ravel()) / np.linalg.norm(x_ref.ravel()) <= 1e-8, (spin, colour)
        _cache[("x3", spin, colour)] = x_ref  # reused by the batched test below


def test_fullsize_config3_twelve_columns_batched(tmw):
    """configs[3] again, the 12 columns in ONE tmw_solve_multi call: every column's exact full-lattice
    residual through the oracle's D, columns (0,0) and (2,1) against the oracle's solution, and one column against the
    single-column solve of the same library."""
    cfg, U = config_fields(3)
    F = config_F(3)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        b = torch.zeros((12, T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        for c in range(12):
            b[c, 0, 0, 0, 0, c // 3, c % 3] = 1.0
        x = torch.empty_like(b)
        infos = ctx.solve_multi(12, b, x, 1e-10)
        xs = x.cpu().numpy()
        x1 = torch.empty_like(x[0])
        ctx.solve(b[5], x1, 1e-10)
        assert float(torch.linalg.vector_norm(x1 - x[5]) / torch.linalg.vector_norm(x1)) <= 1e-8
        del b, x, x1
    torch.cuda.empty_cache()
    for c in range(12):
        assert infos[c]["true_resid"] <= 1e-10 and infos[c]["iters"] > 0
        assert exact_residual(U, F, synth.point_source(L, T, c // 3, c % 3), xs[c], m, c_sw) <= 1e-10, c
    for spin, colour in ORIGIN_COLS:
        x_ref = _cache.get(("x3", spin, colour))
        if x_ref is None:
            x_ref, iref = oracle.bicgstab(U, synth.point_source(L, T, spin, colour), m, c_sw, tol=1e-12, F=F)
            assert iref["status"] == 0
        xg = xs[3 * spin + colour]
        assert np.linalg.norm((xg - x_ref).ravel()) / np.linalg.norm(x_ref.ravel()) <= 1e-8, (spin, colour)


def load_solution_sample(path):
    """tests/golden/cfg4_solution_sample.txt -> (header dict, lexicographic sites, values (n, 4, 3) complex)"""
    hdr, sites, vals = {}, [], []
    with open(path) as f:
        for line in f:
            if line.startswith("#"):
                tok = line[1:].split()
                for k in ("L", "T", "m_re", "m_im", "c_sw", "eps", "xnorm_full_lattice"):
                    if k in tok:
                        hdr[k] = float(tok[tok.index(k) + 1])
                continue
            t = line.split()
            sites.append(int(t[0]))
            vals.append([float(v) for v in t[1:]])
    v = np.array(vals, dtype=np.float64).reshape(len(sites), 12, 2)
    return hdr, np.array(sites, dtype=np.int64), (v[..., 0] + 1j * v[..., 1]).reshape(-1, 4, 3)


def test_fullsize_config4_solve(tmw):
    """configs[4] (48^3 x 144, the benchmark config): tmw_solve of the point source. (i) exact full-lattice residual
    through the oracle's D <= 1e-10; (ii) the solution against the ORACLE's solution at the sampled sites of
    tests/golden/cfg4_solution_sample.txt (the neighbourhood of the source, where the solution lives, corner sites
    and random sites): relative L2 over the sample <= 1e-8, and every sampled site within 1e-8 |x| absolutely;
    (iii) more columns than fit are solved chunk by chunk, a forced unchunked call fails cleanly with TMW_ENOMEM."""
    cfg, U = config_fields(4)
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    b = synth.point_source(L, T, 0, 0)
    dU = torch.from_numpy(U).cuda()
    with tmw.Context(L, T, dU, m, c_sw) as ctx:
        del dU
        x = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        db = torch.from_numpy(b).cuda()
        # 16 columns need 16 x 18.3 GB of workspace here: more than the GPU has. With chunking disabled the call must fail
        # with TMW_ENOMEM before it touches b or x (so one-column buffers are enough), release what it allocated, and
        # leave the context usable.
        ctx.set_debug(tmw.DEBUG_NO_CHUNK)
        with pytest.raises(tmw.TmwError) as e:
            ctx.solve_multi(16, db, x, 1e-10)
        assert e.value.code == tmw.ENOMEM
        ctx.set_debug(0)
        info = ctx.solve(db, x, 1e-10)
        xg = x.cpu().numpy()
        del x
        # with chunking, more columns than fit are solved chunk after chunk: 8 columns = 147 GB of workspace
        n = 8
        bm = torch.zeros((n, T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        for c in range(n):
            bm[c, 0, 0, 0, 0, c // 3, c % 3] = 1.0
        xm = torch.empty_like(bm)
        infos = ctx.solve_multi(n, bm, xm, 1e-10)
        assert all(i["true_resid"] <= 1e-10 and i["iters"] > 0 for i in infos)
        assert float(torch.linalg.vector_norm(xm[0] - torch.from_numpy(xg).cuda()) / torch.linalg.vector_norm(xm[0])) <= 1e-8
        x7 = xm[7].cpu().numpy()
        del bm, xm, db
    torch.cuda.empty_cache()
    assert info["true_resid"] <= 1e-10
    F = config_F(4)
    assert exact_residual(U, F, b, xg, m, c_sw) <= 1e-10
    assert exact_residual(U, F, synth.point_source(L, T, 2, 1), x7, m, c_sw) <= 1e-10
    hdr, sites, ref = load_solution_sample(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg4_solution_sample.txt"))
    assert (hdr["L"], hdr["T"], hdr["m_re"], hdr["m_im"], hdr["c_sw"], hdr["eps"]) == (L, T, m.real, m.imag, c_sw, cfg["eps"])
    got = xg.reshape(-1, 4, 3)[sites]
    assert np.linalg.norm((got - ref).ravel()) / np.linalg.norm(ref.ravel()) <= 1e-8
    # the sample holds the bulk of the solution (it decays fast away from the source), so its norm is the scale of x
    assert np.linalg.norm(ref.ravel()) >= 0.99 * hdr["xnorm_full_lattice"]
    assert np.max(np.abs(got - ref)) <= 1e-8 * hdr["xnorm_full_lattice"]
    _cache.clear()
