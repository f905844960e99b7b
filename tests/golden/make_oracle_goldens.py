#!/usr/bin/env python
"""Writes tests/golden/oracle_neff.txt: effective indices retrieved by the CPU ORACLE ALONE for BASELINE.json's
configs 1, 3 and 4 (n_eff = eta / k0, eps_eff = n_eff^2: PAPER.md:54, :64; pole search Eq. 6-10, PAPER.md:64-95;
tensor entry <-> (direction, polarisation) by DESIGN.md reading R14; two-stage mesh by reading R16).

    python tests/golden/make_oracle_goldens.py [--only cfg1,cfg3,cfg4,dirs,tetra,cfg5b] [--threads T]

(cfg5b - BASELINE config 5b, one 63^3 solve - writes tests/golden/oracle_cfg5b_63.txt and is not in the default set.)

Calls only oracle/ and the seeded input generators (paper_1501_01752_b200/workloads.py, which holds none of the
method's arithmetic).  Nothing here touches the CUDA path.  Existing keys of other groups are kept, so one group can
be regenerated alone.  cfg4 (31^3 orders, O(n^2) Toeplitz product inside full GMRES) takes ~0.5-1 h of host time.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
OUT = os.path.join(HERE, "oracle_neff.txt")
TWO_PI = 2.0 * np.pi

HEADER = """# Effective indices retrieved by the CPU oracle alone (oracle/gsm_oracle.py: retrieve_two_stage over its own solves).
# Written by tests/golden/make_oracle_goldens.py; never edited by hand, never produced by the CUDA path.
# n_eff = eta/k0, eps_eff = n_eff^2 (PAPER.md:54, :64); pole search Eq. 6-10 (PAPER.md:64-95, readings R11-R16);
# tensor entry <-> (propagation axis, polarisation) by reading R14; k0 = 2 pi (lambda = 1).
# key   value
"""


def read_existing():
    vals = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            for line in f:
                line = line.split("#")[0].strip()
                if line:
                    k, v = line.split()
                    vals[k] = v
    return vals


def write_all(vals):
    with open(OUT, "w") as f:
        f.write(HEADER)
        for k in sorted(vals):
            f.write(f"{k} {vals[k]}\n")


def retrieve(orc, geo, c, direction, pol_axis, n_lo, n_hi, dense, tol=1e-13, max_iters=200):
    """Oracle two-stage retrieval along the unit vector `direction` with amplitude e_{pol_axis}."""
    pol = np.zeros(3, dtype=complex)
    pol[pol_axis] = 1.0
    d = np.asarray(direction, dtype=float)
    iters = []

    def xi(kappa):
        out = np.zeros(len(kappa), dtype=complex)
        for i, kv in enumerate(kappa):
            kb = kv * d
            if dense:
                E = orc.solve_dense(c, geo.periods, geo.orders, kb, TWO_PI, geo.eps_b, pol)
            else:
                E, _, it = orc.solve_gmres(c, geo.periods, geo.orders, kb, TWO_PI, geo.eps_b, pol, tol=tol,
                                           max_iters=max_iters, matvec=orc.toeplitz_matvec_c)
                iters.append(it)
            out[i] = orc.zero_order(E)[pol_axis]
        return out
    n, eps, zeta = orc.retrieve_two_stage(xi, TWO_PI, n_lo, n_hi)
    return n, eps, zeta, iters


def put(vals, key, n, eps, zeta):
    vals[key + "_neff_re"] = repr(float(n.real))
    vals[key + "_neff_im"] = repr(float(n.imag))
    vals[key + "_eps_re"] = repr(float(eps.real))
    vals[key + "_zeta_re"] = repr(float(zeta.real))
    vals[key + "_zeta_im"] = repr(float(zeta.imag))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="cfg1,cfg3,cfg4,dirs")
    ap.add_argument("--threads", type=int, default=0)
    args = ap.parse_args()
    if args.threads > 0:
        os.environ["OMP_NUM_THREADS"] = str(args.threads)
    from paper_1501_01752_b200.build import build_oracle
    build_oracle()
    from oracle import gsm_oracle as orc
    from paper_1501_01752_b200 import workloads as wl
    groups = set(args.only.split(","))
    vals = read_existing()
    t0 = time.time()

    if "cfg1" in groups:      # BASELINE config 1: 7^3 sphere lattice, k || z, a = x; dense LU at every point
        geo = wl.sphere_lattice((7, 7, 7))
        c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
        n, eps, zeta, _ = retrieve(orc, geo, c, (0, 0, 1), 0, 1.02, 1.30, dense=True)
        put(vals, "cfg1_7_zx", n, eps, zeta)
        write_all(vals)
        print(f"cfg1 done {time.time() - t0:.0f} s: n = {n}", flush=True)

    if "cfg3" in groups:      # BASELINE config 3: 15^3 ellipsoid lattice, the three diagonal entries (R14)
        geo = wl.ellipsoid_lattice((15, 15, 15))
        c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
        for key, (pa, qa) in wl.DIRECTIONS.items():
            d = np.zeros(3); d[pa] = 1.0
            n, eps, zeta, its = retrieve(orc, geo, c, d, qa, 1.02, 1.30, dense=False)
            put(vals, f"cfg3_15_{key}", n, eps, zeta)
            write_all(vals)
            print(f"cfg3 {key} done {time.time() - t0:.0f} s: n = {n}, iters {min(its)}..{max(its)}", flush=True)

    if "dirs" in groups:      # direction sweep: off-axis unit vectors at config 1, a = s x z / |s x z|
        geo = wl.sphere_lattice((7, 7, 7))
        c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
        for i, (s, a) in enumerate(wl.direction_sweep(5)):
            pol = np.asarray(a, dtype=complex)
            d = np.asarray(s, dtype=float)

            def xi(kappa, d=d, pol=pol):
                return np.array([np.vdot(pol, orc.zero_order(orc.solve_dense(c, geo.periods, geo.orders, kv * d, TWO_PI,
                                                                                geo.eps_b, pol))) for kv in kappa])
            n, eps, zeta = orc.retrieve_two_stage(xi, TWO_PI, 1.02, 1.30)
            put(vals, f"dirs_7_{i}", n, eps, zeta)
        write_all(vals)
        print(f"dirs done {time.time() - t0:.0f} s", flush=True)

    if "cfg4" in groups:      # BASELINE config 4: 31^3 woodpile, eigenmode search along (z,x), (x,y), (x,z)
        geo = wl.woodpile((31, 31, 31))
        c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
        for key, (pa, qa) in (("zx", (2, 0)), ("xy", (0, 1)), ("xz", (0, 2))):
            d = np.zeros(3); d[pa] = 1.0
            n, eps, zeta, its = retrieve(orc, geo, c, d, qa, 1.25, 1.55, dense=False, tol=1e-12)
            put(vals, f"cfg4_31_{key}", n, eps, zeta)
            write_all(vals)
            print(f"cfg4 {key} done {time.time() - t0:.0f} s: n = {n}, iters {min(its)}..{max(its)}", flush=True)

    if "tetra" in groups:     # PAPER.md:127, :143 (Fig. 4): tetragonal lattice of air cavities, 7^3 orders, dense LU
        def line(geo, c, d, pol):
            pol = np.asarray(pol, dtype=complex)

            def xi(kappa):       # reading R28: projection of the 0-th order field on the amplitude
                return np.array([np.vdot(pol, orc.zero_order(orc.solve_dense(c, geo.periods, geo.orders, kv * d, TWO_PI,
                                                                                geo.eps_b, pol))) for kv in kappa])
            return orc.retrieve_two_stage(xi, TWO_PI, TETRA_WINDOW[0], TETRA_WINDOW[1])
        dirs, pols = wl.normal_surface_lines(4)
        for ratio in (0.7, 1.3):     # both sheets of the normal surface in the xz plane
            geo = wl.tetragonal_cavities(ratio)
            c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
            for i in range(len(dirs)):
                n, eps, zeta = line(geo, c, dirs[i], pols[i])
                put(vals, f"tetra_{ratio:g}_surf_{i}", n, eps, zeta)
                print(f"tetra {ratio:g} line {i} done {time.time() - t0:.0f} s: n = {n}", flush=True)
            write_all(vals)
        for ratio in (0.7, 0.85, 1.0, 1.15, 1.3):   # period sweep at constant filling (Fig. 4a): k || z, a = x and a = y
            geo = wl.tetragonal_cavities(ratio)
            c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
            for nm, pol in (("ax", [1.0, 0, 0]), ("ay", [0, 1.0, 0])):
                n, eps, zeta = line(geo, c, np.array([0.0, 0.0, 1.0]), pol)
                put(vals, f"tetra_{ratio:g}_kz_{nm}", n, eps, zeta)
                print(f"tetra sweep {ratio:g} {nm} done {time.time() - t0:.0f} s: n = {n}", flush=True)
            write_all(vals)

    if "cfg5b" in groups:     # BASELINE config 5b: one solve at 63^3 orders on the config-5 voxel composite
        write_cfg5b(orc, wl, t0)


TETRA_WINDOW = (1.39, 1.46)     # n_MG = 1.4213; the anisotropy splits the sheets by a few 1e-3


CFG5B_OUT = os.path.join(HERE, "oracle_cfg5b_63.txt")
CFG5B_SAMPLES = 4096


def write_cfg5b(orc, wl, t0):
    """The oracle's full GMRES (tol 1e-13, O(n^2) Toeplitz product in plain C) for ONE (k, omega) point at 63^3 orders:
    k = (0, 0, 1.12 k0), k0 = 2 pi, a = x.  Stores the 0-th order response, ||E||_2, the iteration count and a seeded
    sample of the field's entries (flat index into E[3][63][63][63], re, im).  About 60 applies of 1.9e11 complex
    multiply-adds each: 20-40 minutes on 8-16 cores."""
    geo = wl.voxel_composite((63, 63, 63), nv=128)
    c = orc.coeffs_voxel(geo.voxels, geo.orders, geo.eps_b)
    kb, k0, pol = np.array([0.0, 0.0, 1.12 * TWO_PI]), TWO_PI, np.array([1.0, 0.0, 0.0], dtype=complex)
    napply = [0]

    def mv(cc, x):
        napply[0] += 1
        print(f"cfg5b apply {napply[0]} at {time.time() - t0:.0f} s", flush=True)
        return orc.toeplitz_matvec_c(cc, x)

    E, hist, iters = orc.solve_gmres(c, geo.periods, geo.orders, kb, k0, geo.eps_b, pol, tol=1e-13, max_iters=150, matvec=mv)
    r = orc.incident(geo.orders, pol) - orc.apply_operator(c, E, geo.periods, kb, k0, geo.eps_b, orc.toeplitz_matvec_c)
    true_res = float(np.linalg.norm(r) / np.linalg.norm(orc.incident(geo.orders, pol)))
    xi = orc.zero_order(E)
    flat = E.ravel()
    idx = np.sort(np.random.default_rng(wl.SEED + 63).choice(flat.size, CFG5B_SAMPLES, replace=False))
    with open(CFG5B_OUT, "w") as f:
        f.write("# BASELINE config 5b: oracle GMRES solution at 63^3 orders (voxel composite of config 5, nv = 128),\n"
                "# k = (0, 0, 1.12 k0), k0 = 2 pi, a = x, tol 1e-13.  Written by tests/golden/make_oracle_goldens.py --only cfg5b\n"
                "# from oracle/ alone; never edited by hand, never produced by the CUDA path.\n"
                "# header lines: key value; then `sample <flat index into E[3][63][63][63]> <re> <im>`\n")
        f.write(f"iters {iters}\n")
        f.write(f"estimated_rel_resid {float(hist[-1])!r}\n")
        f.write(f"true_rel_resid {true_res!r}\n")
        f.write(f"norm_E {float(np.linalg.norm(flat))!r}\n")
        for a in range(3):
            f.write(f"xi{a}_re {float(xi[a].real)!r}\nxi{a}_im {float(xi[a].imag)!r}\n")
        for i in idx:
            f.write(f"sample {int(i)} {float(flat[i].real)!r} {float(flat[i].imag)!r}\n")
    print(f"cfg5b done {time.time() - t0:.0f} s: {iters} iterations, true residual {true_res:.2e}, xi = {xi}", flush=True)


if __name__ == "__main__":
    main()
