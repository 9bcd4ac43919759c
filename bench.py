"""bench.py — the hot path of arXiv:2201.09004 Eqs. (1)-(3) on B200, through the C ABI of include/tmw.h.

    python bench.py --gpus N --steps K --warmup W            (N > 1: launched by torch.distributed.run, one rank per GPU)
    python bench.py --impl reference ...                      (the fp64 CPU oracle as it stands, on the host cores)

Workload (BASELINE.json configs[4], the configuration its metric is quoted on): 48^3 x 144 twisted-mass clover,
m_cri+omega = -0.0398, c_sw = 1.0349, eps = 0.3 seeded random SU(3) links (stand-in for the MILC06 ensemble of
PAPER.md:41 Table 1, which is not available), fp32 12-real gauge. One STEP is one pass of the per-source hot path:
  (i)  tmw_solve of a point source at the origin (mixed-precision even-odd BiCGStab to 1e-10),
  (ii) the Dslash-only run: --napply back-to-back applications of the fp32 hopping block H_{p pbar} (A3),
       ping-ponging even -> odd -> even between two packed parity spinors.
The once-per-gauge-field rows A0-A2 (layout, clover-leaf F, block inverses = tmw_create) are timed separately
and reported as setup_ms. `value` is the Dslash throughput in GFLOP/s at the conventional 1320 flop/site;
`solve_ms` is the BiCGStab time-to-solution. N > 1: replicas only — every rank owns a full context
and takes its own right-hand-side columns (paper_2201_09004_b200/columns.py, round-robin); no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1320          # 8 x (12 + 2 x 66) + 7 x 24, the conventional Wilson Dslash count
BYTES_COMPULSORY = 576        # fp32, 12-real: 96 (in, each site once) + 8 x 48 (links) + 96 (out) per output site
BYTES_STREAMING = 1248        # 8 x 96 + 8 x 48 + 96: no neighbour reuse (the QUDA-style "effective bandwidth" model)


def kernel_bytes_per_site(clover: bool, twisted: bool, reconstruct: int = 12) -> dict:
    """Algorithmic (compulsory: every datum once) bytes per parity site and column of every kernel kind of the solver
    (kinds = include/tmw.h TMW_K_*). fp32 spinor 96 B, fp64 192 B; 8 links: fp32 12-real 384 B (18-real 576),
    fp64 18-real 1152 B; both chirality blocks of the clover term or its inverse: fp32 288 B, fp64 576 B."""
    s32, s64 = 96, 192
    l32, l64 = 8 * 4 * reconstruct, 8 * 144
    c32, c64 = (288, 576) if clover else (0, 0)
    cinv32, cinv64 = (c32 * (2 if twisted else 1), c64 * (2 if twisted else 1))  # twisted clover: (C^2+mu^2)^-1 and C
    return {
        "hop32": s32 + l32 + s32,
        "k1_32": s32 + l32 + cinv32 + s32,
        "k2_32": s32 + l32 + c32 + s32 + s32 + s32,        # in, links, A, aux, out, rhat (the fused <rhat, v>)
        "k2_32_dots": s32 + l32 + c32 + s32 + s32 + s32,   # the same traffic: <t,s>, <t,t>, <rhat,t>, <rhat,s> ride along
        "hop64": s64 + l64 + s64,
        "k1_64": s64 + l64 + cinv64 + s64,
        "k2_64": s64 + l64 + c64 + s64 + s64,
        "xpay64": s64 + l64 + s64 + s64,
        "ainvxpay64": s64 + l64 + cinv64 + s64 + s64,
        "update_s": 3 * s32,
        "update_xrp": 8 * s32,                              # x, p, s, t, v read; x, r, p written
        "acc_y": 2 * s32 + 2 * s64,
        "resid_convert": 3 * s64 + 2 * s32,                 # bhat, Mhat y, r64 | rhat, r (the p fix-up of a mid-run update adds 3 x 96)
        "convert": s64 + s32,
        "dot_norm64": s64,
        "sub_norm": 3 * s64,
        "diag64": s64 + cinv64 + s64,
        "pack_both": 4 * s64,                               # canonical in (both parities), packed out
        "unpack_both": 4 * s64,
    }


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tmw", choices=["tmw", "reference"])
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default 4: 48^3 x 144)")
    ap.add_argument("--napply", type=int, default=200, help="Dslash applications per step")
    ap.add_argument("--e2e-steps", type=int, default=2, help="timed host-buffer steps for the e2e figure")
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--cpu-sites", type=int, default=0, help="oracle sample size in sites (0: sized for ~15 s)")
    ap.add_argument("--multi-rhs", type=int, default=3,
                    help="columns of the extra tmw_solve_multi / tmw_apply_multi leg (0 or 1: skip); 3 fit at 48^3 x 144")
    ap.add_argument("--cpu-solve", action="store_true",
                    help="time the oracle's full-lattice fp64 BiCGStab on this config's source to convergence (6 min at 48^3 x 144 on "
                         "16 cores) instead of the default bounded sample of --cpu-solve-iters iterations")
    ap.add_argument("--cpu-solve-iters", type=int, default=2, help="iterations of the oracle's BiCGStab in the bounded sample (0: skip)")
    ap.add_argument("--domains", default="1x2", help="domain-decomposition leg: domains_z x domains_t (e.g. 1x2, 2x2; 1x1: skip)")
    ap.add_argument("--kernel-reps", type=int, default=20, help="launches per kernel kind in the per-kernel roofline loop (0: skip)")
    ap.add_argument("--stage", type=int, default=0, help="tmw_options.stage: 1 = shared-memory staged fp32 stencil wherever a tile fits (default 0: off)")
    ap.add_argument("--stage-tile", default="0,0,0", help="tmw_options.stage_tile: tile extents x/2,y,z of the staged stencil (0,0,0: chosen by the library)")
    ap.add_argument("--delta", type=float, default=0.0, help="tmw_options.delta: reliable-update threshold (0: the library default 1e-5)")
    ap.add_argument("--columns-per-thread", type=int, default=0, help="tmw_options.columns_per_thread of the multi-column stencil (0: automatic)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--skip-solve", action="store_true",
                    help="profiling aid: steps run only the Dslash part (the JSON line then says so; not a bench value)")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons of one GPU through NVML while the timed region runs."""

    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.mem_samples, self.reason_bits, self.power = [], [], 0, []
        self.timeline = []  # (host perf_counter, SM MHz, reason bits) of every sample
        self.stop_flag = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # NVML missing: the clocks key says so
            self.err = str(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                bits = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.samples.append(mhz)
                self.mem_samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_MEM))
                self.reason_bits |= bits
                self.timeline.append((time.perf_counter(), mhz, bits))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self.stop_flag.wait(self.period)

    def window(self, t_lo: float, t_hi: float):
        """(median SM MHz, share of the samples with sw_power_cap set, samples) over the host-time window [t_lo, t_hi]"""
        w = [(mhz, bits) for (t, mhz, bits) in self.timeline if t_lo <= t <= t_hi]
        if not w:
            return None, None, 0
        return float(np.median([a for a, _ in w])), float(np.mean([1.0 if b & 0x4 else 0.0 for _, b in w])), len(w)

    def summary(self):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + getattr(self, "err", "")]}
        reasons = [name for bit, name in self.REASONS.items() if self.reason_bits & bit and name != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": float(self.max_mhz),
                "mem_mhz": float(np.median(self.mem_samples)) if self.mem_samples else None,
                "reasons": reasons, "samples": len(self.samples),
                "power_w_max": float(max(self.power)) if self.power else None}


def shared_gauge(cfg, rank: int, world: int, barrier):
    """The seeded gauge field of the config as a canonical complex128 array. With several ranks on one node rank 0
    generates it once into /dev/shm and the others map it read-only (replicas share one field)."""
    from paper_2201_09004_b200 import synth
    L, T = cfg["L"], cfg["T"]
    if world == 1:
        return synth.gauge_field(L, T, cfg["eps"], seed=1), None
    path = f"/dev/shm/tmw_bench_gauge_{os.environ.get('MASTER_PORT', '0')}_{L}x{T}.bin"
    shape = (4, T, L, L, L, 3, 3)
    if rank == 0:
        U = synth.gauge_field(L, T, cfg["eps"], seed=1)
        mm = np.memmap(path, dtype=np.complex128, mode="w+", shape=shape)
        mm[...] = U
        mm.flush()
        del mm
        barrier()
        return U, path
    barrier()
    return np.memmap(path, dtype=np.complex128, mode="r", shape=shape), path


def time_oracle_sample(U, psi, cfg, n_sites: int, passes: int = 1):
    """The oracle as it stands on a bounded sample of the workload: (D psi)(x) with the hopping + mass terms of Eq. (2)
    at n_sites sites spread evenly over the lattice (its per-site routine; c_sw = 0 so that one site = the 8 hops
    the GPU metric counts). Returns (seconds, sites, threads)."""
    import oracle
    L, T = cfg["L"], cfg["T"]
    V = L ** 3 * T
    stride = max(1, V // n_sites)
    sites = np.arange(0, V, stride, dtype=np.int64)[:n_sites]
    m = complex(*cfg["m"])
    oracle.apply_sites(U, psi, sites[:1024], m, 0.0)  # page in
    t0 = time.perf_counter()
    for _ in range(passes):
        oracle.apply_sites(U, psi, sites, m, 0.0)
    return time.perf_counter() - t0, int(sites.size) * passes, oracle.num_threads()


def config_dict(cfg, args, world: int, step: str) -> dict:
    """the `config` object of the JSON line: the same keys and values from both arms (the driver compares them)"""
    L, T = cfg["L"], cfg["T"]
    Vh = L ** 3 * T // 2
    return {"workload": cfg["name"], "L": L, "T": T, "m": list(cfg["m"]), "c_sw": cfg["c_sw"], "eps": cfg["eps"],
            "gauge": "fp32 12-real (fp64 18-real for the outer residual)",
            "source": "Z2 noise, seed 2" if cfg["source"] == "z2" else "point, origin",
            "tol": args.tol, "napply": max(2, args.napply // 2 * 2),
            "parallelism": "replicas" if world > 1 else "single",
            "l2": "inputs larger than L2 (a parity spinor is %.0f MB, gauge %.0f MB)" % (Vh * 96 / 1e6, Vh * 8 * 48 / 1e6)}


def run_reference(args, cfg, rank: int):
    """--impl reference: the oracle timed on the host cores, same metric / unit / config; rank 0 only."""
    if rank != 0:
        return
    from paper_2201_09004_b200 import synth
    import oracle
    L, T = cfg["L"], cfg["T"]
    U = synth.gauge_field(L, T, cfg["eps"], seed=1)
    psi = synth.gaussian_spinor(L, T, seed=3)
    n = min(args.cpu_sites or L ** 3 * T, L ** 3 * T)  # default: one pass over the whole lattice per step (1.5 s at 48^3 x 144)
    for _ in range(args.warmup):
        time_oracle_sample(U, psi, cfg, max(1024, n // 8))
    secs, sites = 0.0, 0
    for _ in range(args.steps):
        dt, ns, threads = time_oracle_sample(U, psi, cfg, n)
        secs += dt
        sites += ns
    gflops = FLOP_PER_SITE * sites / secs / 1e9
    sample = (f"oracle.apply_sites (fp64, hopping + mass of Eq. (2)) at {n} evenly spaced sites of the "
              f"{L}^3x{T} field per step")
    line = {"impl": "reference", "metric": "dslash_gflops", "value": gflops, "unit": "GFLOP/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, args, 1, f"{n} sites of oracle.apply_sites per step (the oracle arm has no solve part)"),
            "cpu_baseline": {"value": gflops, "unit": "GFLOP/s", "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": gflops, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "step": f"{n} sites of oracle.apply_sites", "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_tmw(args, cfg, rank: int, world: int, local_rank: int):
    import torch
    from paper_2201_09004_b200 import synth, tmw

    tmw.load()  # raises when libtmw.so is missing: there is no fallback path
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (use --impl reference for the CPU oracle)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(v: float) -> float:
        if dist is None:
            return v
        t = torch.tensor([v], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    L, T, m, c_sw = cfg["L"], cfg["T"], complex(*cfg["m"]), cfg["c_sw"]
    V = L ** 3 * T
    Vh = V // 2
    U, shm_path = shared_gauge(cfg, rank, world, barrier)
    stream = torch.cuda.current_stream().cuda_stream
    ev = lambda: torch.cuda.Event(enable_timing=True)

    # ---- setup rows A0-A2 (once per gauge field): tmw_create from a device-resident canonical gauge field ----
    dU = torch.from_numpy(np.asarray(U)).cuda() if U.flags.writeable else torch.from_numpy(np.array(U)).cuda()
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record()
    tuning = dict(stage=args.stage, stage_tile=tuple(int(v) for v in args.stage_tile.split(",")), columns_per_thread=args.columns_per_thread,
                  delta=args.delta)
    ctx = tmw.Context(L, T, dU, m, c_sw, stream=stream, **tuning)
    e1.record()
    torch.cuda.synchronize()
    setup_ms = e0.elapsed_time(e1)
    del dU
    torch.cuda.empty_cache()
    barrier()
    if shm_path and rank == 0:
        os.unlink(shm_path)

    # ---- inputs resident in HBM: a point source for the solve, a Gaussian spinor for the Dslash-only run ----
    from paper_2201_09004_b200 import columns
    spin, colour = columns.spin_colour(columns.columns_for_rank(rank, world)[0])
    if cfg["source"] == "z2":  # configs[1]: Z2 noise (C15); the others: a point source at the origin (C13)
        b = torch.from_numpy(synth.z2_source(L, T, 2)).cuda()
    else:
        b = torch.zeros((T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        b[0, 0, 0, 0, spin, colour] = 1.0
    x = torch.empty_like(b)
    psi_host = synth.gaussian_spinor(L, T, seed=3)
    nb = ctx.spinor_bytes(tmw.F32)
    pe, po, pe2 = (torch.empty(nb, dtype=torch.uint8, device="cuda") for _ in range(3))
    x.copy_(torch.from_numpy(psi_host))
    ctx.pack(tmw.F32, tmw.EVEN, x, pe)
    torch.cuda.synchronize()

    def dslash_run(n):
        # even -> odd -> even: pe is never overwritten, so the values stay bounded however long the run is
        for i in range(n // 2):
            ctx.apply(tmw.D, tmw.ODD, tmw.F32, pe, po)
            ctx.apply(tmw.D, tmw.EVEN, tmw.F32, po, pe2)

    napply = max(2, args.napply // 2 * 2)
    infos = []

    def step(timers):
        s0, s1, d0, d1 = ev(), ev(), ev(), ev()
        s0.record()
        info = None if args.skip_solve else ctx.solve(b, x, args.tol)
        s1.record()
        d0.record()
        dslash_run(napply)
        d1.record()
        timers.append((s0, s1, d0, d1))
        infos.append(info)

    for _ in range(max(3, args.warmup)):
        step([])
    sampler = ClockSampler(local_rank)
    timers = []
    barrier()
    sampler.start()
    launches0 = ctx.launch_count()
    counts0 = ctx.kernel_counts()
    t0, t1 = ev(), ev()
    torch.cuda.synchronize()
    host_t0 = time.perf_counter()  # the device is idle: t0 fires now, so device offsets from t0 map onto the host clock
    t0.record()
    for _ in range(args.steps):
        step(timers)
    t1.record()
    barrier()
    sampler.stop_flag.set()
    launches = ctx.launch_count() - launches0
    counts1 = ctx.kernel_counts()
    total_ms = max_over_ranks(t0.elapsed_time(t1))
    solve_ms = [a.elapsed_time(bb) for a, bb, _, _ in timers]
    dsl_ms = [c.elapsed_time(d) for _, _, c, d in timers]
    dsl_total_ms = max_over_ranks(sum(dsl_ms))
    solve_mean_ms = max_over_ranks(sum(solve_ms) / len(solve_ms))
    info = infos[-1] or {"iters": None, "reliable_updates": None, "true_resid": None}
    sites = float(Vh) * napply * args.steps * world
    gflops = FLOP_PER_SITE * sites / (dsl_total_ms * 1e-3) / 1e9
    # SURVEY 8(d) protocol: the Dslash part of every step is one repeat of `napply` back-to-back launches; the roofline
    # figure is the MEDIAN repeat (min and every repeat with the SM clock it ran at are printed beside it)
    per_launch_ms = [v / napply for v in dsl_ms]
    repeats = []
    for (_, _, d0, d1), v in zip(timers, per_launch_ms):
        lo, hi = host_t0 + t0.elapsed_time(d0) * 1e-3, host_t0 + t0.elapsed_time(d1) * 1e-3
        mhz, capped, nsamp = sampler.window(lo, hi) if sampler.ok else (None, None, 0)
        repeats.append({"ms_per_launch": v, "sm_mhz": mhz, "power_capped_share": capped, "clock_samples": nsamp})
    dsl_median_ms, dsl_min_ms = float(np.median(per_launch_ms)), float(min(per_launch_ms))
    capped = [r["power_capped_share"] for r in repeats if r["power_capped_share"] is not None]
    regime = None if not capped else ("power-capped" if float(np.median(capped)) >= 0.5 else "burst")
    t_launch_s = dsl_median_ms * 1e-3  # this rank's median-repeat launch duration, events on `stream`
    peak, peak_src = load_peaks()
    achieved = BYTES_COMPULSORY * Vh / t_launch_s / 1e9
    # ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, by kernel kind (profiles/kernel_traffic.csv, one
    # `ncu --set full` capture per kind; the .md beside it has the commands)
    traffic_by_kind = {}
    tp = os.path.join(ROOT, "profiles", "kernel_traffic.csv")
    if os.path.exists(tp):
        import csv
        with open(tp) as f:
            for row in csv.DictReader(f):
                if row["workload"] == cfg["name"] and int(row["columns"]) == 1:
                    traffic_by_kind[row["kind"]] = float(row["dram_bytes_per_launch"])
    traffic = traffic_by_kind.get("hop32")
    roofline = {"bound": "hbm", "kernel": "dslash_kernel<float,12,EPI_HOP> (fp32 hopping block, A3)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "peak_source": peak_src, "bytes_per_site": BYTES_COMPULSORY, "sites_per_launch": Vh,
                "launch_ms": 1e3 * t_launch_s, "streaming_model_gbs": BYTES_STREAMING * Vh / t_launch_s / 1e9,
                "frac_of_8TBs_nominal": achieved / 8000.0,
                "statistic": f"median of {len(per_launch_ms)} repeats of {napply} launches", "regime": regime,
                "frac_min_repeat": BYTES_COMPULSORY * Vh / (dsl_min_ms * 1e-3) / 1e9 / peak,
                "frac_mean": BYTES_COMPULSORY * Vh / (sum(dsl_ms) * 1e-3 / (napply * args.steps)) / 1e9 / peak}

    # ---- the whole solve against the roofline: algorithmic bytes of ONE tmw_solve = (column applications of every kernel
    # kind the context issued inside the timed region, tmw_kernel_counts) x (bytes per site of that kind) x V_h,
    # + the solver's memsets and device copies, over solve_ms ----
    bps = kernel_bytes_per_site(c_sw != 0.0, c_sw != 0.0 and m.imag != 0.0)
    roofline_solve, roofline_kernels = None, None
    if not args.skip_solve:
        per_solve = {k: (counts1[k] - counts0[k]) / args.steps for k in counts1}
        per_solve["hop32"] -= napply  # the Dslash-only part of the step is not the solve
        by_kind = {k: per_solve[k] * bps[k] * Vh for k in bps if per_solve.get(k)}
        other = 2.0 * per_solve["copy_bytes"] + per_solve["memset_bytes"]  # a copy reads and writes
        solve_bytes = sum(by_kind.values()) + other
        t_solve = sum(solve_ms) / len(solve_ms) * 1e-3
        ach = solve_bytes / t_solve / 1e9
        roofline_solve = {"bound": "hbm", "kernel": "tmw_solve: all kernels of one mixed-precision even-odd BiCGStab solve (A3-A8)",
                          "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None, "peak_source": peak_src,
                          "algorithmic_gb": solve_bytes / 1e9, "solve_ms": 1e3 * t_solve,
                          "column_applications_per_solve": {k: v for k, v in per_solve.items() if v and not k.endswith("_bytes")},
                          "gb_by_kind": {k: v / 1e9 for k, v in sorted(by_kind.items(), key=lambda kv: -kv[1])},
                          "memset_and_copy_gb": other / 1e9,
                          "uncounted": "the 1-thread scalar kernels and the per-iteration 2 KB scalar download (no field traffic)"}
        # ---- every kernel the solve spends time in, alone: CUDA events around back-to-back launches on the context stream
        # (tmw_time_kernel), on the vectors the solve left in the workspaces ----
        if args.kernel_reps > 0:
            roofline_kernels = {}
            kinds = ["hop32", "k1_32", "k2_32", "k2_32_dots", "update_s", "update_xrp", "k1_64", "k2_64", "hop32_loadonly"]
            for kind in kinds:
                ms = ctx.time_kernel(kind, args.kernel_reps)
                nbytes = bps["hop32" if kind == "hop32_loadonly" else kind] * Vh
                a_k = nbytes / (ms * 1e-3) / 1e9
                roofline_kernels[kind] = {"bound": "hbm", "achieved": a_k, "peak": peak, "unit": "GB/s", "frac": a_k / peak,
                                          "traffic": traffic_by_kind.get(kind), "launch_ms": ms,
                                          "bytes_per_site": bps["hop32" if kind == "hop32_loadonly" else kind], "sites_per_launch": Vh,
                                          "share_of_solve": (per_solve.get(kind, 0.0) * ms / (1e3 * t_solve)) if kind != "hop32_loadonly" else None}

    # ---- e2e: the same two calls with HOST buffers (pinned), host<->device copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        cbytes = V * 24 * 8
        hb = b.cpu().pin_memory()
        hx = torch.empty((T, L, L, L, 4, 3), dtype=torch.complex128).pin_memory()
        hpsi = torch.from_numpy(psi_host).pin_memory()
        ctx.set_location(tmw.HOST)
        es, ea = [], []
        n_e2e = max(1, args.e2e_steps)
        for i in range(1 + n_e2e):  # one untimed pass first (allocates the staging buffers)
            a0, a1, a2 = ev(), ev(), ev()
            barrier()
            a0.record()
            ctx.solve(hb.data_ptr(), hx.data_ptr(), args.tol)
            a1.record()
            ctx.apply(tmw.D, tmw.FULL, tmw.F64, hpsi.data_ptr(), hx.data_ptr())
            a2.record()
            torch.cuda.synchronize()
            if i > 0:
                es.append(a0.elapsed_time(a1))
                ea.append(a1.elapsed_time(a2))
        ctx.set_location(tmw.DEVICE)
        apply_ms = max_over_ranks(sum(ea) / len(ea))
        e2e = {"value": FLOP_PER_SITE * float(V) * world / (apply_ms * 1e-3) / 1e9, "unit": "GFLOP/s",
               "h2d_bytes_per_step": 2 * cbytes, "d2h_bytes_per_step": 2 * cbytes,
               "call": "tmw_apply(TMW_D, TMW_FULL) with HOST pointers: canonical fp64 spinor in (H2D), D psi out (D2H)",
               "apply_ms": apply_ms, "solve_ms": max_over_ranks(sum(es) / len(es)),
               "solve_call": "tmw_solve with HOST pointers: b in (H2D), x out (D2H)", "steps": n_e2e}
        del hb, hx, hpsi

    # ---- several right-hand sides in one call (the "12 columns" of PAPER.md:78): reported beside the
    # single-column figures, outside the timed step. Columns = as many of this rank's propagator columns as fit. ----
    multi = None
    if args.multi_rhs > 1 and not args.skip_solve:
        n = args.multi_rhs
        mine = columns.columns_for_rank(rank, world)
        bm = torch.zeros((n, T, L, L, L, 4, 3), dtype=torch.complex128, device="cuda")
        for c in range(n):
            sp, co = columns.spin_colour((mine[0] + c) % columns.N_COLUMNS)
            bm[c, 0, 0, 0, 0, sp, co] = 1.0
        xm = torch.empty_like(bm)
        pm = torch.empty(nb * n, dtype=torch.uint8, device="cuda")
        pm2 = torch.empty_like(pm)
        for c in range(n):
            pm[c * nb:(c + 1) * nb].copy_(pe)
        m0, m1, m2, m3 = ev(), ev(), ev(), ev()
        nsch = max(2, napply // 8)
        for i in range(2):  # first pass untimed (grows the workspaces)
            barrier()
            k0 = ctx.kernel_counts()
            m0.record()
            minfos = ctx.solve_multi(n, bm, xm, args.tol)
            m1.record()
            for _ in range(napply // 2):
                ctx.apply_multi(tmw.D, tmw.ODD, tmw.F32, n, pm, pm2)
            m2.record()
            for _ in range(nsch):
                ctx.apply_schur_multi(tmw.D, tmw.F32, n, pm, pm2)
            m3.record()
            torch.cuda.synchronize()
            k1 = ctx.kernel_counts()
        ms_solve = max_over_ranks(m0.elapsed_time(m1))
        ms_hop = max_over_ranks(m1.elapsed_time(m2)) / (napply // 2)
        ms_schur = max_over_ranks(m2.elapsed_time(m3)) / nsch
        multi = {"nrhs": n, "solve_ms_per_rhs": ms_solve / n, "solve_iters": [i["iters"] for i in minfos],
                 "solve_reliable_updates": [i["reliable_updates"] for i in minfos],
                 "solve_true_resid_max": max(i["true_resid"] for i in minfos),
                 "dslash_ms_per_rhs": ms_hop / n, "dslash_gflops": FLOP_PER_SITE * float(Vh) * n * world / (ms_hop * 1e-3) / 1e9,
                 "call": "tmw_solve_multi / tmw_apply_multi, columns resident in HBM"}
        # roofline of the multi-column hop launch: per site and column 96 B in + 96 B out + 384 B of links shared by n
        bpc = 192.0 + 384.0 / n
        ach = bpc * Vh * n / (ms_hop * 1e-3) / 1e9
        pk, pk_src = load_peaks()
        staged = (k1["staged"] - k0["staged"]) > 0
        multi["roofline"] = {"bound": "hbm", "kernel": ("dslash_stage_kernel" if staged else "dslash_kernel") + "<float,12,EPI_HOP,NR=2|3> (multi-column hop)",
                             "achieved": ach, "peak": pk, "unit": "GB/s", "frac": ach / pk, "bytes_per_site_and_column": bpc, "peak_source": pk_src,
                             "note": "not HBM-bound: the links are amortised, the 8 neighbour spinors per column are not (DESIGN.md 6b)"}
        # K1 + K2 (one Schur-operator application) on n columns: per site and column K1 96 in + 96 out, K2 96 in + 96 aux + 96 out,
        # + the links of both launches and the two clover fields shared by the n columns
        bps_schur = 5 * 96.0 + (bps["k1_32"] - 2 * 96.0 + bps["k2_32"] - 4 * 96.0) / n  # shared: links x 2, C^-1 (K1), C (K2)
        ach_s = bps_schur * Vh * n / (ms_schur * 1e-3) / 1e9
        multi["schur_ms_per_rhs"] = ms_schur / n
        multi["roofline_schur"] = {"bound": "hbm", "kernel": "K1 + K2 on %d columns (tmw_apply_schur_multi, fp32)" % n, "achieved": ach_s, "peak": pk,
                                   "unit": "GB/s", "frac": ach_s / pk, "bytes_per_site_and_column": bps_schur, "peak_source": pk_src}
        multi["tuning"] = {"stage": args.stage, "stage_tile": args.stage_tile, "columns_per_thread": args.columns_per_thread,
                           "staged_kernel_ran": staged}
        # the fp32 ALU ceiling beside it (register-only FMA loops, tmw_time_kernel): with the links amortised the multi-column hop
        # is as close to this ceiling as to the HBM one
        try:
            fmas = float(tmw.FFMA_PROBE_FMAS_PER_THREAD) * 256 * 8 * torch.cuda.get_device_properties(local_rank).multi_processor_count
            t_f, t_f2 = ctx.time_kernel("ffma_probe", 5), ctx.time_kernel("ffma2_probe", 5)
            peak_tf = 2 * fmas / (min(t_f, t_f2) * 1e-3) / 1e12
            multi["alu"] = {"bound": "alu", "achieved": multi["dslash_gflops"] / world / 1e3, "peak": peak_tf, "unit": "TFLOP/s",
                            "frac": multi["dslash_gflops"] / world / 1e3 / peak_tf, "ffma_tflops": 2 * fmas / (t_f * 1e-3) / 1e12,
                            "ffma2_tflops": 2 * fmas / (t_f2 * 1e-3) / 1e12,
                            "note": "achieved = 1320 flop/site of the hop at the multi-column rate; peak = measured register-only fp32 FMA rate "
                                    "(2 flop per FMA); ~45 % of the kernel's fp32 instructions are adds and multiplies that count 1 flop"}
        except tmw.TmwError:
            pass
        del bm, xm, pm, pm2
        torch.cuda.empty_cache()

    # ---- domain decomposition: the same calls on a context cut into domains on THIS GPU: what the face
    # pack / copy / interior / exterior split costs when there is no second GPU to gain from (reported beside the undivided
    # figures, outside the timed step) ----
    dd = None
    pz, pt = (int(v) for v in args.domains.lower().split("x"))
    if pz * pt > 1 and not args.skip_solve:
        from paper_2201_09004_b200 import domains as dom
        part = dom.Partition(L, T, pz, pt)
        dUd = torch.from_numpy(np.asarray(U)).cuda() if U.flags.writeable else torch.from_numpy(np.array(U)).cuda()
        dctx = tmw.Context(L, T, dUd, m, c_sw, stream=stream, domains_z=pz, domains_t=pt)
        del dUd
        torch.cuda.empty_cache()
        x.copy_(torch.from_numpy(psi_host))
        dctx.pack(tmw.F32, tmw.EVEN, x, pe)
        d0, d1, d2 = ev(), ev(), ev()
        for i in range(2):
            barrier()
            d0.record()
            dinfo = dctx.solve(b, x, args.tol)
            d1.record()
            for _ in range(napply // 2):
                dctx.apply(tmw.D, tmw.ODD, tmw.F32, pe, po)
            d2.record()
            torch.cuda.synchronize()
        ms_hop = max_over_ranks(d1.elapsed_time(d2)) / (napply // 2)
        dd = {"domains_z": pz, "domains_t": pt, "devices": 1,
              "dslash_ms": ms_hop, "dslash_gflops": FLOP_PER_SITE * float(Vh) * world / (ms_hop * 1e-3) / 1e9,
              "dslash_vs_undivided": ms_hop / (dsl_total_ms / (napply * args.steps)),
              "solve_ms": max_over_ranks(d0.elapsed_time(d1)), "solve_iters": dinfo["iters"], "solve_true_resid": dinfo["true_resid"],
              "exchange_bytes_per_dslash_fp32": part.exchange_bytes(4), "face_bytes_fp32": {"z": part.face_bytes(dom.Z, 4) if part.cut(dom.Z) else 0,
                                                                                        "t": part.face_bytes(dom.T_DIR, 4) if part.cut(dom.T_DIR) else 0},
              "note": "all domains on one GPU: the exchange is a same-device copy; multi-GPU placement unmeasured on hardware"}
        dctx.destroy()
        torch.cuda.empty_cache()

    # ---- the oracle beside it: rank 0, N = 1 only, a bounded sample of the same workload ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n = args.cpu_sites
        if not n:
            dt, ns, _ = time_oracle_sample(U, psi_host, cfg, 100_000)
            n = int(max(100_000, 30.0 * ns / dt))  # sized from a cold 100k-site probe: 10-15 s of oracle work once warm
        passes = max(1, -(-n // V))
        n = min(n, V)
        dt, ns, threads = time_oracle_sample(U, psi_host, cfg, n, passes)
        cpu = {"value": FLOP_PER_SITE * ns / dt / 1e9, "unit": "GFLOP/s", "cores": threads, "kind": "oracle",
               "sample": f"oracle.apply_sites (fp64, hopping + mass of Eq. (2), explicit 4x4 gamma matrices) at {n} "
                         f"evenly spaced sites of the same {L}^3x{T} field, {passes} pass(es), {dt:.1f} s",
               "msites_per_s": ns / dt / 1e6}
        # the oracle's BiCGStab beside tmw_solve (the paper's one number for this path is a CPU BiCGStab time):
        # to convergence with --cpu-solve, else a bounded sample: runs of --cpu-solve-iters - 1 and --cpu-solve-iters iterations
        # (each = 2 D applications + the recurrences on the full lattice), reported per iteration
        cpu["note"] = ("not like for like: the oracle is a deliberately plain fp64 program (explicit 4x4 gamma matrices on full spinors, 18-real "
                       "links, AoS, no even-odd, no SIMD), the GPU figure is the fp32 spin-projected 12-real kernel; the reference ships no CPU code")
        if (args.cpu_solve or args.cpu_solve_iters > 0) and not args.skip_solve:
            import oracle
            import psutil
            need_gb = V * (4 * 9 + 54 + 9 * 12) * 16 / 1e9  # gauge + F + 9 spinors (complex128)
            avail_gb = psutil.virtual_memory().available / 1e9
            if avail_gb < 1.15 * need_gb:
                cpu.update(solve_s=None, solve=f"skipped: the oracle's BiCGStab needs {need_gb:.0f} GB of host memory, {avail_gb:.0f} GB available")
            else:
                bsrc = synth.z2_source(L, T, 2) if cfg["source"] == "z2" else synth.point_source(L, T, spin, colour)
                t0 = time.perf_counter()
                Fo = oracle.field_strength(np.asarray(U)) if c_sw != 0.0 else None
                t_f = time.perf_counter() - t0
                t0 = time.perf_counter()
                if args.cpu_solve:
                    _, oinfo = oracle.bicgstab(np.asarray(U), bsrc, m, c_sw, tol=args.tol, F=Fo)
                    dt = time.perf_counter() - t0
                    cpu.update(solve_s=dt + t_f, solve_iters=oinfo["iters"], solve_true_resid=oinfo["true_resid"], solve_kind="to convergence",
                               solve="oracle.bicgstab (full-lattice fp64 BiCGStab, no preconditioning) to tol, incl. its clover-leaf setup "
                                     f"({t_f:.1f} s)")
                else:
                    # two bounded runs of k1 < k2 iterations; their difference is the cost of k2 - k1 iterations with the
                    # start-up and the closing true-residual application cancelled. Nothing is extrapolated: the line carries
                    # the measured seconds per iteration, not a product with an iteration count taken from elsewhere.
                    k2 = max(2, args.cpu_solve_iters)
                    k1 = k2 - 1
                    t0 = time.perf_counter()
                    oracle.bicgstab(np.asarray(U), bsrc, m, c_sw, tol=1e-300, max_iter=k1, F=Fo)
                    dt1 = time.perf_counter() - t0
                    t0 = time.perf_counter()
                    oracle.bicgstab(np.asarray(U), bsrc, m, c_sw, tol=1e-300, max_iter=k2, F=Fo)
                    dt2 = time.perf_counter() - t0
                    per_iter = (dt2 - dt1) / (k2 - k1)
                    cpu.update(solve_s=None, solve_kind="bounded sample, per iteration", solve_sample_s=dt1 + dt2, solve_sample_iters=[k1, k2],
                               solve_s_per_iter=per_iter, solve_fixed_s=dt1 - k1 * per_iter, solve_setup_s=t_f,
                               solve=f"oracle.bicgstab (full-lattice fp64 BiCGStab, no preconditioning): runs of {k1} and {k2} iterations timed "
                                     f"({dt1:.1f} s, {dt2:.1f} s); solve_s_per_iter = their difference, solve_fixed_s = start-up + closing "
                                     f"residual, solve_setup_s = its clover-leaf setup; no whole-solve figure is derived (solve_s null). "
                                     "--cpu-solve runs it to convergence (340 s measured at 48^3 x 144 to 1e-10: "
                                     "profiles/r2_oracle_cfg4_solve.md)")
                del Fo

    ctx.destroy()
    if rank == 0:
        line = {"metric": "dslash_gflops", "value": gflops, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": config_dict(cfg, args, world, ""),
                "step": ("SOLVE SKIPPED (profiling run, not a bench value): " if args.skip_solve else
                         f"1 tmw_solve(tol={args.tol:g}) + ") + f"{napply} fp32 Dslash applications",
                "dslash_gsites_per_s": sites / (dsl_total_ms * 1e-3) / 1e9, "dslash_ms": dsl_total_ms / (napply * args.steps),
                "dslash_ms_median": dsl_median_ms, "dslash_ms_min": dsl_min_ms, "dslash_repeats": repeats,
                "solve_ms": solve_mean_ms, "solve_iters": info["iters"], "solve_reliable_updates": info["reliable_updates"],
                "solve_true_resid": info["true_resid"], "setup_ms": setup_ms,
                "roofline": roofline, "roofline_solve": roofline_solve, "roofline_kernels": roofline_kernels,
                "cpu_baseline": cpu, "e2e": e2e, "multi_rhs": multi, "domain_decomposition": dd, "gpu_launches": int(launches),
                "clocks": sampler.summary()}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse_args()
    from paper_2201_09004_b200 import synth
    cfg = synth.CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torch.distributed.run --nproc-per-node {args.gpus}")
    run_tmw(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
