"""Writes tests/golden/cfg4_solution_sample.txt: the ORACLE's solution of BASELINE.json configs[4] at a fixed sample
of sites, for tests/test_gpu_fullsize.py::test_fullsize_config4_solve.

    python tests/golden/make_cfg4_solution_sample.py            (needs ~48 GB of host memory, 20-40 min on 8 cores)

Imports only oracle/ and the seeded input generators (paper_2201_09004_b200.synth holds no method arithmetic); nothing
here touches the CUDA path. What is solved: D x = b on the 48^3 x 144 lattice, D of PAPER.md:62 Eq. (2) + :67 Eq. (3)
with m_cri + omega = -0.0398, c_sw = 1.0349 (Table 1), eps = 0.3 seed-1 synthetic SU(3) links (stand-in for
the MILC06 ensemble), b = point source at the origin, spin 0, colour 0 (the first of the "12 columns"), by
the oracle's full-lattice fp64 BiCGStab (no preconditioning) to |r|/|b| <= 1e-12.

Sample: every site within L1 distance 3 of the source (where the solution lives: it decays by ~10 per hop on these
rough fields), the 4^4 sites nearest to the lattice corners (all kinds of boundary wrap), and 800 seeded random sites.
File format: '#' header lines (parameters, iterations, the oracle's own true residual, the full-lattice |x|_2), then one
line per site: lexicographic index (x fastest) and the 24 reals of x(site) in (spin, colour, re/im) order, %.17e.
"""
from __future__ import annotations

import itertools
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2201_09004_b200 import synth  # noqa: E402

OUT = os.path.join(HERE, "cfg4_solution_sample.txt")
N_RANDOM, SEED, RADIUS, TOL = 800, 404, 3, 1e-12


def sample_sites(L: int, T: int) -> np.ndarray:
    lex = lambda x, y, z, t: (x % L) + L * ((y % L) + L * ((z % L) + L * (t % T)))
    s = []
    r = range(-RADIUS, RADIUS + 1)
    for dx, dy, dz, dt in itertools.product(r, r, r, r):
        if abs(dx) + abs(dy) + abs(dz) + abs(dt) <= RADIUS:
            s.append(lex(dx, dy, dz, dt))
    edge, tedge = [0, 1, L - 2, L - 1], [0, 1, T - 2, T - 1]
    for t, z, y, x in itertools.product(tedge, edge, edge, edge):
        s.append(lex(x, y, z, t))
    s += list(np.random.default_rng(SEED).integers(0, L ** 3 * T, size=N_RANDOM))
    return np.unique(np.array(s, dtype=np.int64))


def main(idx: int = 4) -> None:
    cfg = synth.CONFIGS[idx]
    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    t0 = time.time()
    U = synth.gauge_field(L, T, cfg["eps"], seed=1)
    F = oracle.field_strength(U)
    b = synth.point_source(L, T, 0, 0)
    print(f"fields ready after {time.time() - t0:.0f} s", flush=True)
    x, info = oracle.bicgstab(U, b, m, c_sw, tol=TOL, F=F)
    print(f"solved after {time.time() - t0:.0f} s: {info}", flush=True)
    assert info["status"] == 0 and info["true_resid"] <= 10 * TOL
    sites = sample_sites(L, T)
    vals = x.reshape(-1, 12)[sites].view(np.float64).reshape(len(sites), 24)
    xnorm = float(np.linalg.norm(x.ravel()))
    with open(OUT + ".tmp", "w") as f:
        f.write("# Oracle solution of BASELINE.json configs[4] at sampled sites; written by tests/golden/make_cfg4_solution_sample.py\n")
        f.write("# (imports only oracle/ and the seeded input generators). D of PAPER.md:62 Eq. (2) + :67 Eq. (3); parameters of\n")
        f.write("# Table 1 (PAPER.md:41); point source at the origin, spin 0, colour 0 (PAPER.md:78).\n")
        f.write(f"# L {L} T {T} m_re {m.real!r} m_im {m.imag!r} c_sw {c_sw!r} eps {cfg['eps']!r} gauge_seed 1\n")
        f.write(f"# solver oracle.bicgstab tol {TOL:g} iters {info['iters']} true_resid {info['true_resid']:.3e}\n")
        f.write(f"# xnorm_full_lattice {xnorm:.17e}\n")
        f.write(f"# sites {len(sites)} = L1-ball radius {RADIUS} around the source + 4^4 corner sites + {N_RANDOM} random (seed {SEED})\n")
        for s, v in zip(sites, vals):
            f.write(str(int(s)) + " " + " ".join(f"{a:.17e}" for a in v) + "\n")
    os.replace(OUT + ".tmp", OUT)
    print(f"wrote {OUT} ({len(sites)} sites) after {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    main()
