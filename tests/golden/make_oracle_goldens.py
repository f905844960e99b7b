#!/usr/bin/env python
"""Writes tests/golden/oracle_neff.txt: effective indices retrieved by the CPU ORACLE ALONE for BASELINE.json's
configs 1, 3 and 4 (n_eff = eta / k0, eps_eff = n_eff^2: PAPER.md:54, :64; pole search Eq. 6-10, PAPER.md:64-95;
tensor entry <-> (direction, polarisation) by DESIGN.md reading R14; two-stage mesh by reading R16).

    python tests/golden/make_oracle_goldens.py [--only cfg1,cfg3,cfg4,dirs] [--threads T]

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


if __name__ == "__main__":
    main()
