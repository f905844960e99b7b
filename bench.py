#!/usr/bin/env python
"""bench.py - throughput of the GSM hot path on B200 (BASELINE.json metric: (k, omega) solves/s and operator applies/s
at 31^3 orders; % of the HBM roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl gsm|reference]

Workload (BASELINE.json config 5a; recipe in DESIGN.md "Input recipe"): random voxel composite
(20 seeded spheres on a 128^3 voxel grid, cubic Lambda = 0.25 lambda), 31^3 Fourier orders (FFT grid 64^3), 256
concurrent (k, omega) solves per GPU: kappa equidistant on n in [1.05, 1.20], k || z, a = x, GMRES tol 1e-10.
One step = one pass of the whole hot path over that batch: a scan of the 256 points (operator applies, Arnoldi /
Gram-Schmidt, least squares, update, true residual, 0-th order response) by gsm_scan: all 256 points in one lock-step
batch, every one a full GMRES solve from x0 = 0 - a "solve" is the paper's solve, the same work
the CPU oracle and the reference arm do per point, and the same headline as round 1.  (Round 2's headline timed
gsm_scan_mesh instead; it is not comparable and is now the named extra `mesh_scan`: the points form the equidistant
kappa mesh of the method, solved in 5 coarse-to-fine waves (16 + 16 + 32 + 64 + 128), each started from
the pole-aware interpolation of the earlier solutions; every point meets the same tolerance, but most need no
iteration, so its points/s grow with the sampling density.)  Inputs: the per-step working set is
~24 GB of Krylov basis, far above the 126 MB L2, so no L2 flush is needed between timed iterations.

Prints ONE JSON line (rank 0).  `value`: plan resident on the device (coefficient spectrum built), per-launch
profiling OFF.  `e2e`: per step the voxel grid is uploaded from pinned host memory and step a0 re-run
(gsm_plan_set_cell), then the scan (through scan_shard.sharded_scan: this rank's block of the list, host-side gather),
the device->host read of the responses, and the host pole search.  `roofline` / `kernel_ms_per_step`: a SECOND pass of
the same K steps with every launch bracketed by CUDA events on the plan's stream (gsm_plan_profile); algorithmic bytes
are billed from the final iteration counts of every solve.  (In that pass a lock-step batch iterates as one group of
solves; unprofiled it iterates as 2-4 groups on streams of their own, so its kernels overlap and the step is shorter
than the sum of the kernel times.)  `cpu_baseline`: the CPU oracle as it stands (O(n^2)
Toeplitz product + full GMRES) on one of the 256 points, plus one operator apply (the metric's other half).

--impl reference: the oracle itself on the host cores, one solve (one point of the scan) per step.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "(k,omega) solves/s at 31^3 orders, batch 256"
UNIT = "solves/s"
ORDERS = (31, 31, 31)
BATCH = 256
TOL = 1e-10
MAX_ITERS = 64
LEVELS = 1          # headline: plain lock-step gsm_scan, every point from a zero start
MESH_LEVELS = 5     # the `mesh_scan` extra: gsm_scan_mesh waves
N_LO, N_HI = 1.05, 1.20
TWO_PI = 2.0 * np.pi


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def _traffic(kernel, alg_bytes_per_launch):
    """DRAM bytes per launch of `kernel` from the committed `ncu --set full` capture (profiles/ncu_traffic.csv: one row
    per captured launch - first, middle and late iterations - with its dram__bytes_read+write and its algorithmic bytes):
    (sum of captured DRAM bytes / sum of their algorithmic bytes) x this run's average algorithmic bytes per launch.
    None if that kernel was not captured."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        rows = [line.strip().split(",") for line in f if line.strip() and not line.startswith("#")]
    hdr = rows[0]
    dram = alg = 0.0
    for r in rows[1:]:
        if r[hdr.index("kernel")] == kernel:
            dram += float(r[hdr.index("dram_bytes")])
            alg += float(r[hdr.index("algorithmic_bytes")])
    return dram / alg * alg_bytes_per_launch if alg > 0 else None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms (B200_PROFILING.md) from the start of the timed region to
    the end of the profiled second pass (the same steps again): the timed region alone is a few tens of ms."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", str(self.index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(rank, world):
    """The scan list of this rank: BATCH points of a (BATCH * world)-point equidistant kappa mesh whose window grows with
    the number of ranks (rank r scans n in [N_LO + r w, N_LO + (r + 1) w), w = N_HI - N_LO), so that the mesh spacing -
    which decides how good an interpolated guess is - is the same at every N (weak scaling over equal work)."""
    from paper_1501_01752_b200 import workloads as wl
    geo = wl.voxel_composite(ORDERS, nv=128)
    kappa_all = wl.kappa_mesh(N_LO, N_LO + world * (N_HI - N_LO), BATCH * world)
    kappa = kappa_all[rank * BATCH:(rank + 1) * BATCH]
    kb, k0, pol = wl.scan_points(kappa, 2, 0)
    return geo, kappa, kb, k0, pol


def host_cores():
    """Threads the oracle's OpenMP loop can use: the affinity mask of this process."""
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_solve_once(geo, kb, k0, pol):
    """One solve by the CPU oracle as it stands; returns (seconds, iterations, threads)."""
    from oracle import gsm_oracle as orc
    c = orc.coeffs_voxel(geo.voxels, geo.orders, geo.eps_b)
    t0 = time.perf_counter()
    _, hist, iters = orc.solve_gmres(c, geo.periods, geo.orders, kb, float(k0), geo.eps_b, pol[0::2] + 1j * pol[1::2],
                                     tol=TOL, max_iters=MAX_ITERS, matvec=orc.toeplitz_matvec_c)
    return time.perf_counter() - t0, iters, min(orc.num_threads(), host_cores())


def oracle_apply_once(geo, kb, k0, reps=3):
    """Operator applies by the CPU oracle as it stands (O(n^2) Toeplitz product + Green dyadic); seconds per apply."""
    from oracle import gsm_oracle as orc
    from paper_1501_01752_b200 import workloads as wl
    c = orc.coeffs_voxel(geo.voxels, geo.orders, geo.eps_b)
    x = wl.random_field(1, geo.orders)[0]
    orc.apply_operator(c, x, geo.periods, kb, float(k0), geo.eps_b, orc.toeplitz_matvec_c)
    t0 = time.perf_counter()
    for _ in range(reps):
        orc.apply_operator(c, x, geo.periods, kb, float(k0), geo.eps_b, orc.toeplitz_matvec_c)
    return (time.perf_counter() - t0) / reps


def oracle_small_sizes():
    """the oracle as it stands at the smaller configs - one operator apply and one full GMRES solve each
    (7^3 sphere, 1x1x63 laminate, 15^3 ellipsoid); seconds.  63^3 is not run: 1.9e11 complex MACs per apply."""
    from oracle import gsm_oracle as orc
    from paper_1501_01752_b200 import workloads as wl
    out = []
    for name, geo, kbv, k0v in (("7^3 sphere (cfg 1)", wl.sphere_lattice((7, 7, 7)), [0.0, 0.0, 1.2 * TWO_PI], TWO_PI),
                                ("1x1x63 laminate (cfg 2)", wl.laminate(), [0.0, 0.0, 0.9], 0.5),
                                ("15^3 ellipsoid (cfg 3)", wl.ellipsoid_lattice(), [0.0, 0.0, 1.1 * TWO_PI], TWO_PI)):
        c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
        kbv = np.asarray(kbv)
        x = wl.random_field(1, geo.orders)[0]
        orc.apply_operator(c, x, geo.periods, kbv, k0v, geo.eps_b, orc.toeplitz_matvec_c)
        t0 = time.perf_counter()
        orc.apply_operator(c, x, geo.periods, kbv, k0v, geo.eps_b, orc.toeplitz_matvec_c)
        t_apply = time.perf_counter() - t0
        t0 = time.perf_counter()
        _, _, its = orc.solve_gmres(c, geo.periods, geo.orders, kbv, k0v, geo.eps_b, np.array([1.0, 0, 0], dtype=complex),
                                    tol=TOL, max_iters=200, matvec=orc.toeplitz_matvec_c)
        out.append({"workload": name, "apply_s": t_apply, "solve_s": time.perf_counter() - t0, "iters": int(its)})
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from __graft_entry__ import build_oracle
    build_oracle()
    geo, kappa, kb, k0, pol = workload(0, 1)
    times, its, cores = [], [], 1
    for s in range(args.warmup + args.steps):
        p = (s * 37) % BATCH
        t, it, cores = oracle_solve_once(geo, kb[p], k0[p], pol[p])
        if s >= args.warmup:
            times.append(t); its.append(it)
    total = float(np.sum(times))
    value = len(times) / total
    sample = f"1 of the {BATCH} (k,omega) points per step (full GMRES solve, O(n^2) Toeplitz product), mean {np.mean(its):.1f} iterations"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME, "orders": list(ORDERS), "batch": 1, "tol": TOL},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


WORKLOAD_NAME = ("config5a: random voxel composite (20 seeded spheres, 128^3 voxels, Lambda=0.25 lambda), 31^3 orders, "
                 "FFT grid 64^3, 256 concurrent (k,omega) solves per GPU, complex fp64, GMRES tol 1e-10")


def run_gsm(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the GSM hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        dist.barrier()
    from paper_1501_01752_b200 import gsm

    geo, kappa, kb, k0, pol = workload(rank, world)
    stream = torch.cuda.Stream()
    plan = gsm.plan_from_geometry(geo, max_iters=MAX_ITERS, max_batch=BATCH, stream=stream, flags=args.flags)
    pinned_grid = torch.from_numpy(geo.voxels).pin_memory()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def step():
        return plan.scan(kb, k0, pol, tol=TOL, levels=args.levels)

    from paper_1501_01752_b200 import scan_shard, workloads as wl
    kappa_all = wl.kappa_mesh(N_LO, N_LO + world * (N_HI - N_LO), BATCH * world)
    kb_all, k0_all, pol_all = wl.scan_points(kappa_all, 2, 0)

    def step_e2e():
        """What a user of the library runs: new cell -> a0, this rank's block of the scan list, gather, pole search."""
        plan.set_cell(geo.periods, eps_bg=geo.eps_bg, eps_b=geo.eps_b, voxels=pinned_grid)
        resp, iters, resid = scan_shard.sharded_scan(lambda a, b, c: plan.scan(a, b, c, tol=TOL, levels=args.levels)[:3],
                                                     kb_all, k0_all, pol_all, rank, world)
        eta, zeta, best = gsm.pole_search(kappa_all, resp[:, 0], 5, 10)
        return resp, iters, resid, (eta[best] if best >= 0 else None)

    for _ in range(args.warmup):
        resp, iters, resid, st = step()
    assert st >= 0 and float(np.max(resid)) <= 1e-9, f"solve failed: status {st}, max residual {np.max(resid):.2e}"

    # ---- device-resident timed region (per-launch profiling off) ---------------------------------------------------
    sampler = ClockSampler(local)
    plan.profile(False)
    barrier()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = plan.info()["launches"]
    e0.record(stream)
    for _ in range(args.steps):
        resp, iters, resid, st = step()
    e1.record(stream)
    barrier()
    gpu_launches = int(plan.info()["launches"] - launches0)      # every kernel the library enqueued in the timed region
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    value = BATCH * world * args.steps / (ms_total * 1e-3)

    def profiled_pass(levels, nsteps):
        """nsteps more steps of the same scan with a CUDA event pair around every launch: kernel split and bytes."""
        plan.profile(True)
        plan.profile_read(reset=True)
        barrier()
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        q0.record(stream)
        for _ in range(nsteps):
            plan.scan(kb, k0, pol, tol=TOL, levels=levels)
        q1.record(stream)
        barrier()
        pr = plan.profile_read(reset=True)
        plan.profile(False)
        return {k: v for k, v in pr.items() if v[0] > 0 and k != "plan"}, q0.elapsed_time(q1) / nsteps

    def kernel_report(timed, nsteps, peak):
        dom = max(timed, key=lambda k: timed[k][1])
        n_l, ms_l, by_l = timed[dom]
        kernels_ms = sum(v[1] for v in timed.values())
        roof = {"bound": "hbm", "kernel": dom, "achieved": by_l / (ms_l * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                "frac": by_l / (ms_l * 1e-3) / 1e9 / peak, "traffic": _traffic(dom, by_l / n_l), "launches": n_l,
                "avg_launch_ms": ms_l / n_l, "algorithmic_bytes_per_launch": by_l / n_l, "share_of_step": ms_l / kernels_ms}
        if dom == "xy_conv":
            # The plane convolution is not HBM-bound (DRAM 17 %): its roofs are the fp64 pipe and the shared-memory pipe
            # (profiles/xy_conv64_roofs.md).  Report it against the fp64 roof: algorithmic flops 5 P log2 P per line
            # transform + 6 per spectrum multiply, peak = 63.8 fp64 lane-ops/clk/SM measured with a DFMA
            # loop x 148 SMs x 1.965 GHz x 2 flop.
            Wb2, Cb = 2.0 * 16.0 * 3 * 64 * 31 * 31, 16.0 * 64 ** 3
            units = (by_l - Cb * n_l) / Wb2                               # solve-applies billed to the class
            flops = units * 3.0 * (2 * 5 * (31 * 64 + 64 * 64) * 64 * 6 + 6 * 64 ** 3)
            fpeak = 63.8 * 148 * 1.965e9 * 2 / 1e12
            roof.update({"bound": "alu", "achieved": flops / (ms_l * 1e-3) / 1e12, "peak": fpeak, "unit": "TFLOP/s",
                         "frac": flops / (ms_l * 1e-3) / 1e12 / fpeak, "algorithmic_GBps": by_l / (ms_l * 1e-3) / 1e9,
                         "peak_source": "fp64 pipe, measured DFMA loop (DESIGN.md 5); the shared-memory pipe is the one "
                                        "that saturates first in this kernel (72 % at a full batch)",
                         "algorithmic_flops_per_launch": flops / n_l})
        return roof, {k: v[1] / nsteps for k, v in timed.items()}, \
            {k: (v[2] / (v[1] * 1e-3) / 1e9 if v[1] > 0 and v[2] > 0 else None) for k, v in timed.items()}

    # ---- second pass of the headline scan, profiled: the kernel split and the roofline ------------------------------------
    timed, ms_profiled = profiled_pass(args.levels, args.steps)
    clocks = sampler.stop() if rank == 0 else None

    # ---- the same 256 points as an ordered mesh (gsm_scan_mesh: coarse-to-fine waves with interpolated guesses) ------
    plan.scan(kb, k0, pol, tol=TOL, levels=MESH_LEVELS)
    barrier()
    z0, z1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    z0.record(stream)
    for _ in range(3):
        _, z_iters, z_resid, _ = plan.scan(kb, k0, pol, tol=TOL, levels=MESH_LEVELS)
    z1.record(stream)
    barrier()
    z_ms = max_over_ranks(z0.elapsed_time(z1)) / 3
    z_timed, z_ms_profiled = profiled_pass(MESH_LEVELS, 3)

    # ---- a longer list through the same plan: 1024 points, max_batch 256 (waves of the mesh scan are chunked) -------------
    kb4, k04, pol4 = wl.scan_points(wl.kappa_mesh(N_LO, N_HI, 4 * BATCH), 2, 0)
    plan.scan(kb4, k04, pol4, tol=TOL, levels=MESH_LEVELS + 2)
    barrier()
    l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0.record(stream)
    _, l_iters, l_resid, _ = plan.scan(kb4, k04, pol4, tol=TOL, levels=MESH_LEVELS + 2)
    l1.record(stream)
    barrier()
    l_ms = l0.elapsed_time(l1)

    # ---- end to end through the C ABI with host buffers ---------------------------------------------------------
    for _ in range(min(args.warmup, 2)):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        out = step_e2e()
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e_value = BATCH * world * args.steps / e2e_s
    h2d = int(pinned_grid.numel() * 16 + kb.nbytes + k0.nbytes + pol.nbytes + 16)
    # per solve: response (48 B), iterations, residual, active flag, residual-check flag; per lock-step tick: nactive (4 B)
    if args.levels > 1:
        wave_of, _, _ = gsm.mesh_schedule(BATCH, args.levels, 1)
        ticks = sum(int(iters[wave_of == w].max()) + 2 for w in range(int(wave_of.max()) + 1))
    else:
        ticks = int(np.max(iters)) + 2
    d2h = int(resp.nbytes + iters.nbytes + resid.nbytes + 8 * BATCH + 4 * ticks)

    # ---- operator applies/s (the other half of BASELINE.json's metric) -------------------------------------------
    x = torch.randn((BATCH, 3) + ORDERS, dtype=torch.complex128, device="cuda")
    y = torch.empty_like(x)
    torch.cuda.synchronize()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    napply = 20
    with torch.cuda.stream(stream):       # the plan's stream is torch's current stream: no cross-stream ordering needed
        for _ in range(3):
            plan.apply(kb, k0, x, out=y)
        barrier()
        a0.record(stream)
        for _ in range(napply):
            plan.apply(kb, k0, x, out=y)
        a1.record(stream)
    barrier()
    apply_ms = max_over_ranks(a0.elapsed_time(a1)) / napply
    # one solve's apply alone (SURVEY 8(d) "single and batch-256"): x, y, W and Chat (~13 MB) stay in L2
    with torch.cuda.stream(stream):
        for _ in range(3):
            plan.apply(kb[:1], k0[:1], x[:1], out=y[:1])
        barrier()
        a0.record(stream)
        for _ in range(200):
            plan.apply(kb[:1], k0[:1], x[:1], out=y[:1])
        a1.record(stream)
    barrier()
    apply1_ms = a0.elapsed_time(a1) / 200
    V = 16.0 * 3 * geo.n
    chat_bytes = 16.0 * 64 ** 3
    apply_alg_bytes = 2 * V * BATCH + chat_bytes

    # ---- same workload in the H-field formulation (Eq. 5), informational ------------------------
    plan.close()
    del x, y
    torch.cuda.empty_cache()
    plan_h = gsm.plan_from_geometry(geo, max_iters=MAX_ITERS, max_batch=BATCH, stream=stream, formulation=gsm.FORM_H)
    pol_h = np.zeros_like(pol); pol_h[:, 2] = 1.0                    # h = y (transverse to k || z)
    plan_h.scan(kb, k0, pol_h, tol=TOL)
    h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    h0.record(stream)
    for _ in range(2):
        _, h_iters, h_resid, h_st = plan_h.scan(kb, k0, pol_h, tol=TOL)
    h1.record(stream)
    torch.cuda.synchronize()
    h_ms = h0.elapsed_time(h1) / 2
    fft_grid = list(plan_h.info()["fft_grid"])
    plan_h.close()

    def solve_report(p, kbs_, k0s_, pols_, tol, reps, grid_pts):
        """`reps` timed scans of the points given (one lock-step batch, zero start) with profiling off, then one more with a
        CUDA event pair around every launch: time, kernel split, dominant kernel and whole path against the HBM roof
        (SURVEY 8(d) B_solve = (m(m+1)/2 + 3m + 1) V + m |Chat| per solve)."""
        peak_, _ = _peaks()
        nb = len(k0s_)
        p.scan(kbs_, k0s_, pols_, tol=tol)
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record(stream)
        for _ in range(reps):
            _, its_, res_, _ = p.scan(kbs_, k0s_, pols_, tol=tol)
        r1.record(stream)
        torch.cuda.synchronize()
        ms_ = r0.elapsed_time(r1) / reps
        p.profile(True); p.profile_read(reset=True)
        p.scan(kbs_, k0s_, pols_, tol=tol)
        torch.cuda.synchronize()
        pr_ = {k: v for k, v in p.profile_read(reset=True).items() if v[0] > 0 and k != "plan"}
        p.profile(False)
        Vn = 16.0 * 3 * p.n
        b_ = float(np.sum((its_ * (its_ + 1.0) / 2 + 3.0 * its_ + 1.0) * Vn)) + float(np.mean(its_)) * 16.0 * grid_pts
        dom_ = max(pr_, key=lambda k: pr_[k][1])
        kms_ = sum(v[1] for v in pr_.values())
        return {"batch": nb, "ms": ms_, "solves_per_s": nb * 1e3 / ms_, "iters": [int(i) for i in its_],
                "max_true_resid": float(np.max(res_)),
                "path_roofline": {"algorithmic_GBps": b_ / (ms_ * 1e-3) / 1e9, "frac": b_ / (ms_ * 1e-3) / 1e9 / peak_},
                "roofline": {"bound": "hbm", "kernel": dom_, "achieved": pr_[dom_][2] / (pr_[dom_][1] * 1e-3) / 1e9, "peak": peak_,
                             "unit": "GB/s", "frac": pr_[dom_][2] / (pr_[dom_][1] * 1e-3) / 1e9 / peak_, "launches": pr_[dom_][0],
                             "avg_launch_ms": pr_[dom_][1] / pr_[dom_][0], "share_of_step": pr_[dom_][1] / kms_, "traffic": None},
                "profiled_pass_ms": kms_, "launches": int(sum(v[0] for v in pr_.values())),
                "kernel_ms": {k: v[1] for k, v in pr_.items()},
                "kernel_GBps": {k: (v[2] / (v[1] * 1e-3) / 1e9 if v[1] > 0 and v[2] > 0 else None) for k, v in pr_.items()}}

    # ---- config 5b: single solves at 63^3 orders (FFT grid 128^3), informational, rank 0 only ------------------------
    c5b = None
    if rank == 0:
        from paper_1501_01752_b200 import workloads as wl
        geo63 = wl.voxel_composite((63, 63, 63), nv=128)
        p63 = gsm.plan_from_geometry(geo63, max_iters=MAX_ITERS, max_batch=1, stream=stream)
        kb63, pol63 = np.array([0.0, 0.0, 1.12 * TWO_PI]), np.array([1.0, 0, 0], dtype=complex)
        p63.solve(kb63, TWO_PI, pol63, tol=TOL)
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        for _ in range(3):
            _, _, it63, res63, _ = p63.solve(kb63, TWO_PI, pol63, tol=TOL)
        s1.record(stream)
        torch.cuda.synchronize()
        solve_ms = s0.elapsed_time(s1) / 3
        x63 = torch.randn((1, 3, 63, 63, 63), dtype=torch.complex128, device="cuda")
        y63 = torch.empty_like(x63)
        for _ in range(3):
            p63.apply(kb63[None], [TWO_PI], x63, out=y63)
        s0.record(stream)
        for _ in range(50):
            p63.apply(kb63[None], [TWO_PI], x63, out=y63)
        s1.record(stream)
        torch.cuda.synchronize()
        ap_ms = s0.elapsed_time(s1) / 50
        V63 = 16.0 * 3 * 63 ** 3
        c5b = {"workload": "config5b: same composite, 63^3 orders, FFT grid 128^3, one solve at a time",
               "solve_ms": solve_ms, "solves_per_s": 1e3 / solve_ms, "iters": int(it63), "true_resid": float(res63),
               "apply_ms": ap_ms, "applies_per_s": 1e3 / ap_ms,
               "apply_algorithmic_GBps": (2 * V63 + 16.0 * 128 ** 3) / (ap_ms * 1e-3) / 1e9,
               "note": "working set of one apply (x, y, W, Chat ~ 150 MB) is about the size of L2"}
        c5b["single_solve"] = solve_report(p63, kb63[None], np.array([TWO_PI]), pol63[None], TOL, 3, 128 ** 3)
        p63.close()
        del x63, y63
        torch.cuda.empty_cache()
        p63b = gsm.plan_from_geometry(geo63, max_iters=MAX_ITERS, max_batch=8, stream=stream)
        kb8, k08, pol8 = wl.scan_points(wl.kappa_mesh(N_LO, N_HI, 8), 2, 0)
        c5b["batch_of_8"] = solve_report(p63b, kb8, k08, pol8, TOL, 2, 128 ** 3)
        p63b.close()
        torch.cuda.empty_cache()
        # ---- the two large sizes of the paper's Table 1 as single solves (context: PAPER.md:111-115 gives 2.2 s and 114 s
        # on a GTX Titan, the latter with the GMRES basis streamed from host RAM); informational
        large = []
        for N in (128, 256):
            gl = wl.sphere_lattice((N, N, N), period=0.3, radius_frac=0.3, eps=9.0)
            pl_ = gsm.plan_from_geometry(gl, max_iters=40, max_batch=1, stream=stream)
            kbl, poll = np.array([0.0, 0.0, 1.3 * TWO_PI]), np.array([1.0, 0, 0], dtype=complex)
            pl_.solve(kbl, TWO_PI, poll, tol=1e-8)
            s0.record(stream)
            _, _, itl, resl, _ = pl_.solve(kbl, TWO_PI, poll, tol=1e-8)
            s1.record(stream)
            torch.cuda.synchronize()
            large.append({"orders": [N, N, N], "unknowns": 3 * N ** 3, "solve_ms": s0.elapsed_time(s1), "iters": int(itl),
                          "true_resid": float(resl), "device_GB": pl_.info()["device_bytes"] / 1e9,
                          "report": solve_report(pl_, kbl[None], np.array([TWO_PI]), poll[None], 1e-8, 1, (2 * N) ** 3)})
            pl_.close()
            torch.cuda.empty_cache()
        c5b["large_orders_single_solve"] = large

    if world > 1:
        dist.barrier()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class -----------------------------------------------------------------
    peak, peak_src = _peaks()
    roof, k_ms, k_gbs = kernel_report(timed, args.steps, peak)
    roof.setdefault("peak_source", peak_src)
    z_roof, z_k_ms, z_k_gbs = kernel_report(z_timed, 3, peak)
    mean_it = float(np.mean(iters))
    # whole-step figure against SURVEY 8(d)'s B_solve = (m(m+1)/2 + 3m + 1) V + m |Chat| per solve
    # (+ 3 V for a solve started from a guess: the apply that forms r0 = b - A x0 and the read of x0 in the update)
    guessed = BATCH - len(range(0, BATCH, 1 << (args.levels - 1))) if args.levels > 1 else 0
    wave0 = np.arange(BATCH) % (1 << (args.levels - 1)) == 0
    b_solve = (float(np.sum((iters * (iters + 1.0) / 2 + 3.0 * iters + 1.0) * V)) + 3.0 * V * guessed
               + float(np.sum(iters)) / BATCH * chat_bytes)
    path_gbs = b_solve * args.steps / (ms_total * 1e-3) / 1e9
    z_wave0 = np.arange(BATCH) % (1 << (MESH_LEVELS - 1)) == 0
    z_b_solve = (float(np.sum((z_iters * (z_iters + 1.0) / 2 + 3.0 * z_iters + 1.0) * V)) + 3.0 * V * float(np.sum(~z_wave0))
                 + float(np.mean(z_iters)) * chat_bytes)

    # ---- CPU oracle on a bounded sample ---------------------------------------------------------------------------
    cpu_t, cpu_it, cores = oracle_solve_once(geo, kb[0], k0[0], pol[0])
    cpu_apply_t = oracle_apply_once(geo, kb[0], k0[0])
    cpu_small = oracle_small_sizes()
    # SURVEY 8(d) / BASELINE.md 2: one oracle apply at 63^3 orders measured (1.9e11 complex multiply-adds); the 63^3 solve and
    # the 256-solve batch at 31^3 are extrapolated from measured pieces and labelled as such
    cpu_apply63_t = oracle_apply_once(wl.voxel_composite((63, 63, 63), nv=128), np.array([0.0, 0.0, 1.12 * TWO_PI]), TWO_PI, reps=1)
    it63_gpu = c5b["single_solve"]["iters"][0] if c5b else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAME, "orders": list(ORDERS), "fft_grid": fft_grid,
                   "batch_per_gpu": BATCH, "tol": TOL, "max_iters": MAX_ITERS, "mean_iters": mean_it,
                   "scan_driver": (f"gsm_scan_mesh, {args.levels} coarse-to-fine waves with interpolated initial guesses "
                                   "(PAPER.md:101 equidistant mesh)" if args.levels > 1 else "gsm_scan, zero start"),
                   "mean_iters_zero_start_wave": float(np.mean(iters[wave0])),
                   "mean_iters_guessed_waves": float(np.mean(iters[~wave0])) if guessed else None,
                   "max_true_resid": float(np.max(resid)), "parallelism": f"scan list sharded over {world} GPU(s), no collective",
                   "streams": "a lock-step batch of 8+ solves iterates as 2-4 groups on streams of the plan's own "
                              "(forked from / joined to the plan's stream); the timed region is bracketed on the plan's stream",
                   "l2": "working set per step ~24 GB >> 126 MB L2; no flush needed"},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "includes": "voxel grid H2D from pinned memory + a0 (gsm_plan_set_cell) + gsm_scan + response D2H + host pole search"},
        "gpu_launches": gpu_launches,
        "clocks": clocks,
        "roofline": roof,
        "path_roofline": {"algorithmic_GBps": path_gbs, "frac": path_gbs / peak,
                          "definition": "SURVEY 8(d) B_solve summed over the batch / step time (profiling off)"},
        "profiled_pass": {"ms_per_step": ms_profiled,
                          "note": "second pass of the same steps with a CUDA event pair around every launch; "
                                  "roofline, kernel_ms_per_step and kernel_GBps come from it, value and e2e do not. With "
                                  "profiling on, a lock-step batch iterates as one group; without it, as 2-4 groups on "
                                  "streams of their own whose kernels overlap, so the kernel times of this pass add up to "
                                  "more than ms_per_step"},
        "kernel_ms_per_step": k_ms,
        "kernel_GBps": k_gbs,
        "applies_per_s": BATCH * world / (apply_ms * 1e-3),
        "apply": {"ms_per_batch_apply": apply_ms, "algorithmic_GBps": apply_alg_bytes / (apply_ms * 1e-3) / 1e9,
                  "frac": apply_alg_bytes / (apply_ms * 1e-3) / 1e9 / peak, "definition": "(2V x 256 + |Chat|) / time",
                  "single_apply_us": 1e3 * apply1_ms,
                  "single_apply_note": "batch of 1: three launches whose working set (x, y, W, Chat ~ 13 MB) stays in L2; "
                                       "latency-bound, no HBM figure is meaningful (SURVEY 8(d))"},
        "mesh_scan": {"value": BATCH * world / (z_ms * 1e-3), "unit": "mesh points/s", "ms_per_step": z_ms,
                                "mean_iters": float(np.mean(z_iters)), "max_true_resid": float(np.max(z_resid)),
                                "mean_iters_zero_start_wave": float(np.mean(z_iters[z_wave0])),
                                "mean_iters_guessed_waves": float(np.mean(z_iters[~z_wave0])),
                                "note": f"gsm_scan_mesh on the same 256 points, {MESH_LEVELS} coarse-to-fine waves with "
                                        "interpolated initial guesses (PAPER.md:101 equidistant mesh; round 2's headline). "
                                        "NOT comparable with `value`, cpu_baseline or the reference arm: most points are "
                                        "accepted after one verifying apply, so points/s grow with the sampling density",
                                "roofline": z_roof,
                                "path_roofline": {"algorithmic_GBps": z_b_solve / (z_ms * 1e-3) / 1e9,
                                                  "frac": z_b_solve / (z_ms * 1e-3) / 1e9 / peak},
                                "profiled_pass_ms_per_step": z_ms_profiled,
                                "kernel_ms_per_step": z_k_ms, "kernel_GBps": z_k_gbs},
        "scan_1024_points": {"value": 4 * BATCH / (l_ms * 1e-3), "unit": UNIT, "ms": l_ms,
                             "ratio_to_256_point_mesh_scan": l_ms / z_ms,
                             "mean_iters": float(np.mean(l_iters)), "max_true_resid": float(np.max(l_resid)),
                             "note": f"same window, 1024 kappa points, max_batch 256, gsm_scan_mesh with {MESH_LEVELS + 2} waves"},
        "h_form": {"value": BATCH / (h_ms * 1e-3), "unit": UNIT, "ms_per_step": h_ms, "mean_iters": float(np.mean(h_iters)),
                   "max_true_resid": float(np.max(h_resid)), "note": "same workload, Eq. 5 (H-field) formulation, this rank only"},
        "config5b_63cubed": c5b,
        "cpu_baseline": {"value": 1.0 / cpu_t, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"1 of the {BATCH} (k,omega) points (full GMRES solve with the O(n^2) Toeplitz product, "
                                   f"{cpu_it} iterations, {cpu_t:.1f} s)",
                         "applies_per_s": 1.0 / cpu_apply_t,
                         "apply_sample": f"one operator apply at 31^3 orders (O(n^2) Toeplitz product + Green dyadic), "
                                         f"mean of 3, {cpu_apply_t:.2f} s",
                         "gpu_over_oracle_like_for_like": value / world * cpu_t,
                         "ratio_note": "value per GPU / this oracle figure: both are full GMRES solves from x0 = 0 of points of "
                                       "the same list (a GPU-over-slow-CPU figure, not a kernel-quality one)",
                         "other_sizes": cpu_small,
                         "apply_63cubed_s": cpu_apply63_t,
                         "apply_63cubed_sample": "one operator apply at 63^3 orders (config 5b), measured once after one warm-up apply",
                         "solve_63cubed_s_extrapolated": cpu_apply63_t * (it63_gpu + 1) if it63_gpu else None,
                         "solve_63cubed_note": "EXTRAPOLATED: measured apply x (iterations of the GPU solve of the same point + 1)",
                         "batch_256_at_31cubed_s_extrapolated": cpu_t * BATCH,
                         "batch_256_note": "EXTRAPOLATED: the one measured 31^3 solve x 256"},
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gsm", choices=["gsm", "reference"])
    ap.add_argument("--flags", type=int, default=0, help="diagnostic plan flags (include/gsm.h GSM_FLAG_*), for A/B runs")
    ap.add_argument("--levels", type=int, default=LEVELS, help="headline scan: 1 = plain lock-step gsm_scan (default), > 1 = gsm_scan_mesh waves")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gsm(args)


if __name__ == "__main__":
    main()
