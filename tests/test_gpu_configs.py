"""BASELINE.json configs 2, 3 and 4 run on the GPU path AS STATED (64-frequency laminate scan along z and x, TE/TM;
128 (k, omega) points per principal axis of the ellipsoid lattice; eigenmode search along three directions of the 31^3
woodpile), against the CPU oracle; plus the alternative code paths (two-sweep Gram-Schmidt, generic FFT passes,
fused persistent apply) held to the same parity bar through the plan's diagnostic flags.

Bars (BASELINE.json north_star): relative L2 field error <= 1e-9, true Krylov residual <= 1e-10, eps_eff within 1e-8.
Expected effective indices are computed by the oracle in the test, or read from tests/golden/oracle_neff.txt (written by
tests/golden/make_oracle_goldens.py from the oracle alone)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

from conftest import load_golden, load_oracle_golden  # noqa: E402
from oracle import gsm_oracle as orc  # noqa: E402
from paper_1501_01752_b200 import gsm, workloads as wl  # noqa: E402

TWO_PI = 2.0 * np.pi


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def coeffs(geo):
    if geo.voxels is not None:
        return orc.coeffs_voxel(geo.voxels, geo.orders, geo.eps_b)
    return orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)


def scan_lines(plan, lines, meshes, tol):
    """One gsm_scan over the concatenated kappa meshes of many lines (direction, polarisation, k0); returns, per line,
    the response component along the polarisation axis."""
    kb, kk, pol = [], [], []
    for ln, kap in zip(lines, meshes):
        a, b, c = wl.scan_points(kap, ln["prop"], ln["pol"], ln["k0"])
        kb.append(a); kk.append(b); pol.append(c)
    resp, iters, resid, st = plan.scan(np.concatenate(kb), np.concatenate(kk), np.concatenate(pol), tol=tol)
    assert st == gsm.OK and float(resid.max()) <= 1e-10
    out, o = [], 0
    for ln, kap in zip(lines, meshes):
        out.append(resp[o:o + len(kap), ln["pol"]])
        o += len(kap)
    return out


def two_stage_gpu(plan, lines, ncoarse=29, nfine=18, fine_step=0.002, tol=1e-12):
    """The two-stage retrieval of reading R16 for many lines at once: every stage is ONE gsm_scan over all lines;
    gsm_pole_search (host C++) per line.  Returns the list of complex n_eff."""
    coarse = [np.linspace(ln["n_lo"], ln["n_hi"], ncoarse) * ln["k0"] for ln in lines]
    est = []
    for ln, kap, xi in zip(lines, coarse, scan_lines(plan, lines, coarse, tol)):
        eta, zeta, best = gsm.pole_search(kap, xi, 5, 10)
        assert best >= 0, f"no pole in the coarse window of {ln}"
        est.append(eta[best].real)
    fine = [e + fine_step * ln["k0"] * (np.arange(nfine) - 0.5 * (nfine - 1)) for ln, e in zip(lines, est)]
    out = []
    for ln, kap, xi in zip(lines, fine, scan_lines(plan, lines, fine, tol)):
        eta, zeta, best = gsm.pole_search(kap, xi, 5, 10)
        assert best >= 0, f"no pole in the fine window of {ln}"
        out.append(eta[best] / ln["k0"])
    return out


def two_stage_oracle(geo, c, ln, solve):
    pol = np.zeros(3, dtype=complex); pol[ln["pol"]] = 1.0
    d = np.zeros(3); d[ln["prop"]] = 1.0

    def xi(kap):
        return np.array([orc.zero_order(solve(c, geo.periods, geo.orders, kv * d, ln["k0"], geo.eps_b, pol))[ln["pol"]]
                         for kv in kap])
    n, eps, zeta = orc.retrieve_two_stage(xi, ln["k0"], ln["n_lo"], ln["n_hi"])
    return n


# ---- closed forms for the laminate (Rytov; SURVEY 8(c) pins, also used by tests/test_oracle_pins.py) -------------------
def rytov_cos_KL(k0, e1, e2, d1, d2):
    k1, k2 = k0 * math.sqrt(e1), k0 * math.sqrt(e2)
    return math.cos(k1 * d1) * math.cos(k2 * d2) - 0.5 * (k1 / k2 + k2 / k1) * math.sin(k1 * d1) * math.sin(k2 * d2)


def rytov_inplane_beta(k0, e1, e2, d1, d2, tm):
    import scipy.optimize

    def f(beta):
        q1, q2 = np.sqrt(complex(k0 * k0 * e1 - beta * beta)), np.sqrt(complex(k0 * k0 * e2 - beta * beta))
        p = q1 / q2 * ((e2 / e1) if tm else 1.0)
        return (np.cos(q1 * d1) * np.cos(q2 * d2) - 0.5 * (p + 1 / p) * np.sin(q1 * d1) * np.sin(q2 * d2) - 1.0).real
    lo, hi = k0 * math.sqrt(min(e1, e2)) * 1.0001, k0 * math.sqrt(max(e1, e2)) * 0.9999
    return scipy.optimize.brentq(f, lo, hi, xtol=1e-15, rtol=1e-15)


def laminate_lines():
    """BASELINE config 2: 64 frequencies Lambda_z / lambda_j = 0.25 j / 64 (length unit Lambda_z), propagation along z
    (a = x; pass band only, j <= 46: reading R21) and along x with a = y (TE) and a = z (TM).  Coarse windows of about
    +-10 % around the Rytov root (narrower towards the band edge, where the mirror pole 2 pi - K enters), placed so that
    the root falls mid-way between two of the 29 nodes: the TE poles ARE the Rytov roots to ~1e-7, and a sample on a
    pole is a singular system (reading R16)."""
    def window(ref, w):
        lo = ref * (1.0 - w)
        return lo, lo + 28.0 * (ref * w / 13.5)      # node spacing h = ref w / 13.5: ref = lo + 13.5 h
    lines = []
    for j in range(1, 65):
        k0 = TWO_PI * 0.25 * j / 64
        cK = rytov_cos_KL(k0, 1.0, 9.0, 0.5, 0.5)
        if abs(cK) < 1.0:
            K = math.acos(cK)
            w = min(0.1, 0.6 * (math.pi - K) / K)
            lo, hi = window(K / k0, w)
            lines.append(dict(fam="z", j=j, prop=2, pol=0, k0=k0, ref=K / k0, n_lo=lo, n_hi=hi))
        for fam, pa, tm in (("xTE", 1, False), ("xTM", 2, True)):
            n = rytov_inplane_beta(k0, 1.0, 9.0, 0.5, 0.5, tm) / k0
            lo, hi = window(n, 0.1)
            lines.append(dict(fam=fam, j=j, prop=0, pol=pa, k0=k0, ref=n, n_lo=lo, n_hi=hi))
    return lines


def test_config2_laminate_64_frequency_scan_z_and_x_te_tm():
    geo = wl.laminate((1, 1, 63))
    lines = laminate_lines()
    assert sum(ln["fam"] == "z" for ln in lines) == 46 and len(lines) == 46 + 128
    plan = gsm.plan_from_geometry(geo, max_iters=200, max_batch=256)
    n_gpu = two_stage_gpu(plan, lines)
    plan.close()
    c = coeffs(geo)
    for ln, ng in zip(lines, n_gpu):
        no = two_stage_oracle(geo, c, ln, orc.solve_dense)
        assert abs(ng * ng - no * no) <= 1e-8, (ln["fam"], ln["j"])
        assert abs(ng.imag) <= 1e-9
        if ln["fam"] != "xTM":          # TE-like: Rytov dispersion, truncation error ~ N^-3
            assert abs(ng.real / ln["ref"] - 1.0) <= 1e-6, (ln["fam"], ln["j"])
        else:                           # TM under the Laurent rule converges only as 1/N: 0.6 % at N3 = 63
            assert 0.004 <= ng.real / ln["ref"] - 1.0 <= 0.007, (ln["fam"], ln["j"])
    # mean-permittivity limits at the longest wavelength (Lambda_z / lambda = 0.0039)
    by = {(ln["fam"], ln["j"]): ng for ln, ng in zip(lines, n_gpu)}
    assert abs(by[("xTE", 1)].real ** 2 - 5.0) <= 2e-3 and abs(by[("z", 1)].real ** 2 - 5.0) <= 2e-3   # arithmetic mean
    assert abs(by[("xTM", 1)].real ** 2 - 1.8) <= 0.03                                                 # harmonic mean side
    # ... and the 1/N trend of the TM value towards Rytov's, on the GPU path
    errs = []
    for N3 in (15, 31, 63):
        g = wl.laminate((1, 1, N3))
        p = gsm.plan_from_geometry(g, max_iters=200, max_batch=32)
        ln = [l for l in lines if l["fam"] == "xTM" and l["j"] == 32][0]
        wide = dict(ln, n_lo=ln["ref"] * 0.98, n_hi=ln["ref"] * 1.12)
        errs.append(abs(two_stage_gpu(p, [wide])[0].real - ln["ref"]))
        p.close()
    assert errs[0] > errs[1] > errs[2] and 1.6 < errs[0] / errs[1] < 2.6 and 1.6 < errs[1] / errs[2] < 2.6


def test_config3_ellipsoid_128_points_per_axis_full_tensor():
    """BASELINE config 3: 128 (k, omega) points per principal axis in ONE lock-step scan of 384 solves (reading R14 for
    the (direction, polarisation) pairs), pole estimate per axis, fine stage, the three diagonal entries of eps_eff
    against the oracle-written golden values."""
    gold = load_oracle_golden()
    geo = wl.ellipsoid_lattice((15, 15, 15))
    plan = gsm.plan_from_geometry(geo, max_iters=120, max_batch=384)
    lines = [dict(key=key, prop=pa, pol=qa, k0=TWO_PI, n_lo=1.02, n_hi=1.30) for key, (pa, qa) in wl.DIRECTIONS.items()]
    n_gpu = two_stage_gpu(plan, lines, ncoarse=128)
    for ln, n in zip(lines, n_gpu):
        assert abs((n * n).real - gold[f"cfg3_15_{ln['key']}_eps_re"]) <= 1e-8 and abs((n * n).imag) <= 1e-8
        assert abs(n.real - gold[f"cfg3_15_{ln['key']}_neff_re"]) <= 1e-8
    plan.close()


def test_config4_woodpile_31cubed_eigenmode_search_three_directions():
    """BASELINE config 4: gsm_retrieve_neff (two-stage scan + pole search) along (z,x), (x,y), (x,z) at 31^3 orders
    against the oracle's own retrieval (tests/golden/oracle_neff.txt; ~0.5 h of oracle time, hence stored)."""
    gold = load_oracle_golden()
    if not all(f"cfg4_31_{k}_zeta_im" in gold for k in ("zx", "xy", "xz")):
        pytest.skip("tests/golden/oracle_neff.txt has no cfg4 entries yet (run make_oracle_goldens.py --only cfg4)")
    geo = wl.woodpile((31, 31, 31))
    plan = gsm.plan_from_geometry(geo, max_iters=150, max_batch=96)
    keys = (("zx", (2, 0)), ("xy", (0, 1)), ("xz", (0, 2)))
    dirs = np.zeros((3, 3)); pols = np.zeros((3, 3), dtype=complex)
    for i, (key, (pa, qa)) in enumerate(keys):
        dirs[i, pa] = 1.0
        pols[i, qa] = 1.0
    # the three directions together: each stage is one lock-step batch (3 x 29, then 3 x 18 solves)
    n, eps, zeta, ls, st = plan.retrieve_neff_many(dirs, pols, [qa for _, (_, qa) in keys], TWO_PI, 1.25, 1.55, tol=1e-12)
    assert st == gsm.OK and np.all(ls == gsm.OK)
    for i, (key, _) in enumerate(keys):
        assert abs(eps[i].real - gold[f"cfg4_31_{key}_eps_re"]) <= 1e-8 and abs(eps[i].imag) <= 1e-8
        assert abs(n[i].real - gold[f"cfg4_31_{key}_neff_re"]) <= 1e-8
        zo = complex(gold[f"cfg4_31_{key}_zeta_re"], gold[f"cfg4_31_{key}_zeta_im"])
        assert abs(zeta[i] - zo) <= 1e-6 * abs(zo)
    plan.close()


# ---- the general-purpose code paths at the same bar -----------------------------------------------------------------------
FLAG_SETS = [gsm.FLAG_TWO_SWEEP, gsm.FLAG_GENERIC_APPLY, gsm.FLAG_FUSED_APPLY, gsm.FLAG_TWO_SWEEP | gsm.FLAG_GENERIC_APPLY]


@pytest.mark.parametrize("flags", FLAG_SETS)
def test_flagged_paths_config1_vs_dense_lu(flags):
    geo = wl.sphere_lattice((7, 7, 7))
    plan = gsm.plan_from_geometry(geo, max_iters=64, flags=flags)
    kb, k0, pol = np.array([0.0, 0.0, 1.2 * TWO_PI]), TWO_PI, np.array([1.0, 0.0, 0.0], dtype=complex)
    E, hist, iters, resid, st = plan.solve(kb, k0, pol, tol=1e-12)
    ref = orc.solve_dense(coeffs(geo), geo.periods, geo.orders, kb, k0, geo.eps_b, pol)
    assert st == gsm.OK and resid <= 1e-10 and rel(E.cpu().numpy(), ref) <= 1e-9
    plan.close()


@pytest.mark.parametrize("flags", [0] + FLAG_SETS)
def test_flagged_paths_17cubed_vs_oracle_gmres(flags):
    """17^3 orders: 64-point axes (three-launch fast path by default; fused persistent launch / generic passes by flag) and the
    cluster or two-sweep Gram-Schmidt, fields against the oracle's GMRES on the O(n^2) product; a batch of 3 so that the
    ticket queue of the fused apply holds several solves."""
    geo = wl.sphere_lattice((17, 17, 17))
    plan = gsm.plan_from_geometry(geo, max_iters=80, max_batch=3, flags=flags)
    c = coeffs(geo)
    kb = np.array([[0.0, 0.0, 1.2 * TWO_PI], [0.3, -0.2, 1.15 * TWO_PI], [1.25 * TWO_PI, 0.0, 0.0]])
    pol = np.array([[1.0, 0, 0], [0.2, 1.0, 0.1j], [0, 0, 1.0]], dtype=complex)
    fields = torch.empty((3, 3, 17, 17, 17), dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, np.full(3, TWO_PI), pol, tol=1e-12, fields=fields)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    F = fields.cpu().numpy()
    for i in range(3):
        ref, _, oit = orc.solve_gmres(c, geo.periods, geo.orders, kb[i], TWO_PI, geo.eps_b, pol[i], tol=1e-13,
                                      max_iters=120, matvec=orc.toeplitz_matvec_c)
        assert rel(F[i], ref) <= 1e-9 and abs(int(iters[i]) - oit) <= 4
    plan.close()


def test_two_sweep_natural_case_past_the_cluster_cap():
    """63 x 63 x 9 orders: one field vector (107 163 complex numbers) no longer fits a thread-block cluster, so the
    two-sweep Gram-Schmidt kernels run without any flag (with the 128-point xy pass and the generic z passes)."""
    geo = wl.Geometry("slab-of-spheres", (0.25, 0.25, 0.1), (63, 63, 9),
                      [dict(kind=wl.SPHERE, center=(0.02, -0.03, 0.0), size=(0.04, 0, 0), eps=5.0)], 1.0, 1.0, None, ())
    plan = gsm.plan_from_geometry(geo, max_iters=80)
    assert plan.info()["fft_grid"] == (128, 128, 32)
    kb, pol = np.array([0.0, 0.0, 1.1 * TWO_PI]), np.array([1.0, 0.0, 0.0], dtype=complex)
    E, hist, iters, resid, st = plan.solve(kb, TWO_PI, pol, tol=1e-12)
    ref, _, oit = orc.solve_gmres(coeffs(geo), geo.periods, geo.orders, kb, TWO_PI, geo.eps_b, pol, tol=1e-13,
                                  max_iters=120, matvec=orc.toeplitz_matvec_c)
    assert st == gsm.OK and resid <= 1e-10 and rel(E.cpu().numpy(), ref) <= 1e-9 and abs(iters - oit) <= 4
    prof = plan.profile_read()
    assert iters <= prof["sweep_dots"][0] <= iters + 1 and prof["arnoldi_mgs"][0] == 0   # (+ one overlapped launch)
    plan.close()


def test_fused_apply_many_solves_ring_reuse_and_inactive_solves():
    """The fused persistent apply with more solves than ring slots (ring reuse, all three dependency counters) is
    bit-identical to the three-launch apply, also when only some solves of the batch are active (scan with mixed
    convergence goes through the compacted list)."""
    geo = wl.sphere_lattice((19, 17, 18))
    B = 40
    x = torch.from_numpy(wl.random_field(B, geo.orders)).cuda()
    rng = np.random.default_rng(5)
    kb = rng.uniform(-1, 1, (B, 3)) * TWO_PI
    k0 = np.full(B, TWO_PI)
    pf = gsm.plan_from_geometry(geo, max_batch=B, flags=gsm.FLAG_FUSED_APPLY)
    ps = gsm.plan_from_geometry(geo, max_batch=B)
    yf = pf.apply(kb, k0, x).cpu().numpy()
    ys = ps.apply(kb, k0, x).cpu().numpy()
    assert np.array_equal(yf, ys)
    assert pf.profile_read()["apply_fused"][0] == 1 and ps.profile_read()["xy_conv"][0] == 1
    kappa = wl.kappa_mesh(1.02, 1.30, B)
    kbs, kk, pol = wl.scan_points(kappa, 2, 0)
    rf, itf, _, _ = pf.scan(kbs, kk, pol, tol=1e-11)
    rs, its, _, _ = ps.scan(kbs, kk, pol, tol=1e-11)
    assert len(set(itf.tolist())) > 1 and np.array_equal(itf, its) and np.array_equal(rf, rs)
    pf.close(); ps.close()


# ---- Krylov work reused along the kappa mesh --------------------------------------------
def test_scan_guess_on_a_side_stream_is_ordered_with_the_current_stream():
    """Plan.scan / Plan.solve on a plan bound to its own stream: the guesses x0 are produced by a chain of kernels on
    torch's current stream right before the call and the fields are read on it right after, with no manual
    synchronisation.  Same results, bit for bit, as a plan on the current stream."""
    geo = wl.sphere_lattice((17, 17, 17))
    kappa = np.array([1.12, 1.13, 1.14, 1.15]) * TWO_PI
    kb, kk, pol = wl.scan_points(kappa, 2, 0)
    side = torch.cuda.Stream()
    p_side = gsm.plan_from_geometry(geo, max_iters=64, max_batch=4, stream=side)
    p_ref = gsm.plan_from_geometry(geo, max_iters=64, max_batch=4)
    base = torch.empty((4, 3, 17, 17, 17), dtype=torch.complex128, device="cuda")
    p_ref.scan(kb * (1 + 5e-4), kk, pol, tol=1e-10, fields=base)          # neighbouring points' fields as guesses
    torch.cuda.synchronize()
    for rep in range(3):
        x0 = base * 0.0
        for _ in range(20):                       # a chain of kernels on the current stream that produces x0
            x0 = x0 + base / 20.0
        f_side = torch.empty_like(base)
        r1, i1, _, _ = p_side.scan(kb, kk, pol, tol=1e-10, fields=f_side, x0=x0)
        got = f_side.cpu().numpy()                # read on the current stream
        f_ref = torch.empty_like(base)
        r2, i2, _, _ = p_ref.scan(kb, kk, pol, tol=1e-10, fields=f_ref, x0=x0)
        assert np.array_equal(i1, i2) and np.array_equal(r1, r2) and np.array_equal(got, f_ref.cpu().numpy())
        E1 = p_side.solve(kb[0], TWO_PI, [1.0, 0, 0], tol=1e-10)[0].cpu().numpy()
        E2 = p_ref.solve(kb[0], TWO_PI, [1.0, 0, 0], tol=1e-10)[0].cpu().numpy()
        assert np.array_equal(E1, E2)
    p_side.close(); p_ref.close()


def test_scan_guess_matches_oracle_gmres_with_the_same_x0():
    """gsm_scan_guess: GMRES from an initial guess (r0 = b - A x0, E = x0 + d) against the oracle's gmres(x0=...) with the
    SAME x0: the solution of a nearby kappa point, a random field (worse than a zero start: the library falls back to
    the zero start), the exact solution (no iteration), and a slightly scaled exact solution."""
    geo = wl.sphere_lattice((7, 7, 7))
    c = coeffs(geo)
    kappa = np.array([1.12, 1.13, 1.14, 1.15]) * TWO_PI          # away from the pole at 1.0998 (reading R10)
    kb, kk, pol = wl.scan_points(kappa, 2, 0)
    polc = np.array([1.0, 0, 0], dtype=complex)
    exact = [orc.solve_dense(c, geo.periods, geo.orders, kb[i], TWO_PI, geo.eps_b, polc) for i in range(4)]
    near = orc.solve_dense(c, geo.periods, geo.orders, kb[0] * (1 + 5e-4), TWO_PI, geo.eps_b, polc)
    x0 = np.stack([near, wl.random_field(1, geo.orders)[0] * 5.0, exact[2], exact[3] * (1 + 1e-4)])
    plan = gsm.plan_from_geometry(geo, max_iters=64, max_batch=4)
    fields = torch.empty((4, 3, 7, 7, 7), dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, kk, pol, tol=1e-12, fields=fields, x0=torch.from_numpy(x0).cuda())
    r0, it0, _, _ = plan.scan(kb, kk, pol, tol=1e-12)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    F = fields.cpu().numpy()
    for i in range(4):
        assert rel(F[i], exact[i]) <= 1e-9
    ref0, _, oit0 = orc.solve_gmres(c, geo.periods, geo.orders, kb[0], TWO_PI, geo.eps_b, polc, tol=1e-12, x0=x0[0])
    assert rel(F[0], ref0) <= 1e-9 and abs(int(iters[0]) - oit0) <= 2 and iters[0] < it0[0]     # neighbour's field: fewer
    assert iters[1] == it0[1] and np.array_equal(resp[1], r0[1])      # useless guess ignored: identical to the zero start
    assert iters[2] == 0 and np.array_equal(F[2], x0[2])              # exact guess: returned as is
    ref3, _, oit3 = orc.solve_gmres(c, geo.periods, geo.orders, kb[3], TWO_PI, geo.eps_b, polc, tol=1e-12, x0=x0[3])
    assert abs(int(iters[3]) - oit3) <= 2 and iters[3] < it0[3]
    # in place: the guesses sit in the output buffer
    buf = torch.from_numpy(x0).cuda()
    resp2, iters2, _, _ = plan.scan(kb, kk, pol, tol=1e-12, fields=buf, x0=buf)
    assert np.array_equal(iters2, iters) and np.array_equal(buf.cpu().numpy(), F)
    plan.close()


def test_scan_mesh_levels_same_poles_fewer_iterations():
    """gsm_scan_mesh: the equidistant kappa mesh solved coarse to fine with interpolated guesses gives the same fields
    (unique solution; compared with dense LU) and the same pole as the plain scan, in fewer iterations."""
    geo = wl.sphere_lattice((7, 7, 7))
    c = coeffs(geo)
    kappa = wl.kappa_mesh(1.05, 1.20, 45)          # 45 points: ragged against the wave strides; max_batch 16: chunks
    kb, kk, pol = wl.scan_points(kappa, 2, 0)
    plan = gsm.plan_from_geometry(geo, max_iters=64, max_batch=16)
    r1, it1, res1, st1 = plan.scan(kb, kk, pol, tol=1e-12)
    fields = torch.empty((45, 3, 7, 7, 7), dtype=torch.complex128, device="cuda")
    r4, it4, res4, st4 = plan.scan(kb, kk, pol, tol=1e-12, levels=4, fields=fields)
    r0, it0, _, _ = plan.scan(kb, kk, pol, tol=1e-12, levels=1)
    assert st1 == st4 == gsm.OK and np.all(res4 <= 1e-10)
    assert np.array_equal(r0, r1) and np.array_equal(it0, it1)                       # levels = 1 is gsm_scan
    assert it4.sum() < 0.9 * it1.sum() and np.array_equal(it4[::8], it1[::8])        # wave 0 starts from zero
    F = fields.cpu().numpy()
    polc = np.array([1.0, 0, 0], dtype=complex)
    for p in (0, 3, 4, 13, 22, 44):
        ref = orc.solve_dense(c, geo.periods, geo.orders, kb[p], TWO_PI, geo.eps_b, polc)
        if abs(kappa[p] / TWO_PI - 1.0998) > 0.003:       # fields away from the pole (reading R10), xi everywhere
            assert rel(F[p], ref) <= 1e-9
        assert np.array_equal(F[p][:, 3, 3, 3], r4[p])
    e1, z1, b1 = gsm.pole_search(kappa, r1[:, 0], 5, 10)
    e4, z4, b4 = gsm.pole_search(kappa, r4[:, 0], 5, 10)
    assert b1 >= 0 and b4 >= 0 and abs((e4[b4] / TWO_PI) ** 2 - (e1[b1] / TWO_PI) ** 2) <= 1e-8
    plan.close()


# ---- direction sweep at fixed omega -------------------------------------------------
def test_direction_sweep_off_axis_vs_oracle_goldens():
    """gsm_retrieve_neff_many over seeded off-axis propagation directions s (amplitude a = s x z / |s x z|, response =
    projection of the 0-th order field on a) at config 1 / 7^3, all directions in one batch per stage, against the oracle's
    own retrieval with dense LU solves (tests/golden/oracle_neff.txt, group `dirs`)."""
    gold = load_oracle_golden()
    geo = wl.sphere_lattice((7, 7, 7))
    sweep = wl.direction_sweep(5)
    dirs = np.array([s for s, a in sweep]); pols = np.array([a for s, a in sweep], dtype=complex)
    plan = gsm.plan_from_geometry(geo, max_iters=100, max_batch=160)
    n, eps, zeta, ls, st = plan.retrieve_neff_many(dirs, pols, -1, TWO_PI, 1.02, 1.30, tol=1e-12)
    assert st == gsm.OK and np.all(ls == gsm.OK)
    for i in range(5):
        assert abs(n[i].real - gold[f"dirs_7_{i}_neff_re"]) <= 1e-8 and abs(n[i].imag) <= 1e-9
        assert abs(eps[i].real - gold[f"dirs_7_{i}_eps_re"]) <= 1e-8
        zo = complex(gold[f"dirs_7_{i}_zeta_re"], gold[f"dirs_7_{i}_zeta_im"])
        assert abs(zeta[i] - zo) <= 1e-6 * abs(zo)
    assert len({round(float(v.real), 6) for v in n}) > 1          # spatial dispersion: the index depends on the direction
    # a single line gives the same number as the batched call (the solves are independent)
    n1, _, _, st1 = plan.retrieve_neff(dirs[2], pols[2], -1, TWO_PI, 1.02, 1.30, tol=1e-12)
    assert st1 == gsm.OK and abs(n1 - n[2]) <= 1e-10
    with pytest.raises(gsm.GsmError):          # an empty window on any line rejects the call
        plan.retrieve_neff_many(dirs, pols, -1, TWO_PI, [1.02, 1.3, 1.02, 1.02, 1.02], [1.30, 1.2, 1.30, 1.30, 1.30])
    plan.close()


def test_scan_mesh_edge_cases_lossy_hform_short_lists():
    """gsm_scan_mesh where the guess machinery takes its other branches: a lossy inclusion (complex pole, complex
    interpolation weights), the H-form, lists too short for a pole estimate, more levels than the list supports,
    max_batch 1 (every wave in chunks of one), a zero-amplitude point inside the mesh.  The fields must equal the
    plain scan's to the solver tolerance in every case."""
    k0 = TWO_PI
    cases = [
        (wl.sphere_lattice((7, 7, 7), eps=4.0 + 0.3j), gsm.FORM_E, 33, 4, 8),
        (wl.sphere_lattice((5, 5, 5)), gsm.FORM_H, 40, 3, 16),
        (wl.sphere_lattice((5, 5, 5)), gsm.FORM_E, 9, 6, 4),          # 9 points: never enough for the pole search
        (wl.sphere_lattice((5, 5, 5)), gsm.FORM_E, 21, 3, 1),         # one solve at a time
        (wl.sphere_lattice((5, 5, 5)), gsm.FORM_E, 2, 5, 8),
    ]
    for geo, form, npts, levels, mb in cases:
        kappa = wl.kappa_mesh(1.03, 1.25, npts)
        kb, kk, pol = wl.scan_points(kappa, 2, 1 if form == gsm.FORM_H else 0)
        if npts == 21:
            pol[7] = 0.0                                              # zero source in the middle of the mesh
        plan = gsm.plan_from_geometry(geo, max_iters=80, max_batch=mb, formulation=form)
        shape = (npts, 3) + tuple(geo.orders)
        f1 = torch.empty(shape, dtype=torch.complex128, device="cuda")
        f2 = torch.empty(shape, dtype=torch.complex128, device="cuda")
        r1, it1, res1, st1 = plan.scan(kb, kk, pol, tol=1e-12, fields=f1)
        r2, it2, res2, st2 = plan.scan(kb, kk, pol, tol=1e-12, fields=f2, levels=levels)
        assert st1 == st2 == gsm.OK and np.all(res2 <= 1e-10), (geo.name, npts)
        a, b = f1.cpu().numpy(), f2.cpu().numpy()
        for p in range(npts):
            nrm = np.linalg.norm(a[p])
            cond_ok = abs(kappa[p] / k0 - 1.0998) > 0.004 or geo.orders != (7, 7, 7)
            if nrm == 0.0:
                assert np.linalg.norm(b[p]) == 0.0 and it2[p] == 0
            elif cond_ok:
                assert np.linalg.norm(a[p] - b[p]) <= 1e-9 * nrm, (geo.name, npts, p)
        if npts >= 33:            # enough solved points for a pole estimate: the guesses pay (shorter lists: any guess is valid)
            assert it2.sum() < it1.sum()
        plan.close()


def test_scan_slot_refill_bit_identical_and_vs_oracle():
    """GSM_FLAG_SLOT_REFILL: gsm_scan from a zero start with more points than max_batch keeps the lock-step batch full: a slot whose solve has
    finished takes the next pending point, every solve at its own Arnoldi index (the scan is a list
    of independent solves).  Per solve the arithmetic is that of one lock-step batch: bit-identical results; fields
    against the oracle's GMRES; E- and H-form; 64-point fast path (17^3) and generic passes (7^3)."""
    for orders, form in (((17, 17, 17), gsm.FORM_E), ((7, 7, 7), gsm.FORM_E), ((7, 7, 7), gsm.FORM_H)):
        geo = wl.sphere_lattice(orders)
        npts = 11
        kappa = wl.kappa_mesh(1.02, 1.30, npts)
        kb, kk, pol = wl.scan_points(kappa, 2, 0)
        kb[3] = [0.3, -0.2, 1.15 * TWO_PI]                       # one off-axis point with a general amplitude
        pol[3] = [0.2, 0.0, 1.0, 0.0, 0.0, 0.1]
        pol[7] = 0.0                                              # and one zero source (E = 0, no iterations)
        one = gsm.plan_from_geometry(geo, max_iters=80, max_batch=16, formulation=form)
        few = gsm.plan_from_geometry(geo, max_iters=80, max_batch=3, formulation=form, flags=gsm.FLAG_SLOT_REFILL)
        Fa = torch.empty((npts, 3) + orders, dtype=torch.complex128, device="cuda")
        Fb = torch.zeros_like(Fa)
        ra, ia, resa, sta = one.scan(kb, kk, pol, tol=1e-12, fields=Fa)
        rb, ib, resb, stb = few.scan(kb, kk, pol, tol=1e-12, fields=Fb)
        assert sta == gsm.OK and stb == gsm.OK and len(set(ia.tolist())) > 2
        assert np.array_equal(ia, ib) and np.array_equal(ra, rb) and np.array_equal(resa, resb)
        assert torch.equal(Fa, Fb)
        assert ib[7] == 0 and float(Fb[7].abs().max()) == 0.0 and np.all(resb <= 1e-10)
        # without a field buffer the responses are the same
        rc, ic, _, _ = few.scan(kb, kk, pol, tol=1e-12)
        assert np.array_equal(rc, ra) and np.array_equal(ic, ia)
        # launch accounting: the refill scan needs fewer Arnoldi launches than three-at-a-time chunks would
        few.profile_read(reset=True)
        few.scan(kb, kk, pol, tol=1e-12)
        launches = few.profile_read()["arnoldi_mgs"][0]
        chunks = sum(int(ia[p0:p0 + 3].max()) for p0 in range(0, npts, 3))
        assert launches < chunks + 4
        if form == gsm.FORM_E:
            c = coeffs(geo)
            F = Fb.cpu().numpy()
            for p in (3, 10):
                a = pol[p, 0::2] + 1j * pol[p, 1::2]
                if orders[0] == 7:
                    ref = orc.solve_dense(c, geo.periods, geo.orders, kb[p], kk[p], geo.eps_b, a)
                else:
                    ref, _, _ = orc.solve_gmres(c, geo.periods, geo.orders, kb[p], kk[p], geo.eps_b, a, tol=1e-13,
                                                max_iters=120, matvec=orc.toeplitz_matvec_c)
                assert rel(F[p], ref) <= 1e-9
        one.close(); few.close()


def test_scan_slot_refill_max_iters_and_single_slot():
    """Refill with one slot (max_batch 1) and a basis too small to converge: every point stops at max_iters with the best
    iterate and the scan reports GSM_NOT_CONVERGED; with room to converge the single slot reproduces gsm_solve."""
    geo = wl.sphere_lattice((7, 7, 7))
    kappa = wl.kappa_mesh(1.05, 1.25, 5)
    kb, kk, pol = wl.scan_points(kappa, 2, 0)
    short = gsm.plan_from_geometry(geo, max_iters=4, max_batch=2, flags=gsm.FLAG_SLOT_REFILL)
    _, it, res, st = short.scan(kb, kk, pol, tol=1e-12)
    assert st == gsm.NOT_CONVERGED and np.all(it == 4) and np.all(res > 1e-12) and np.all(res < 1.0)
    short.close()
    plan = gsm.plan_from_geometry(geo, max_iters=64, max_batch=1, flags=gsm.FLAG_SLOT_REFILL)
    F = torch.empty((5, 3, 7, 7, 7), dtype=torch.complex128, device="cuda")
    _, it, res, st = plan.scan(kb, kk, pol, tol=1e-12, fields=F)
    assert st == gsm.OK
    for p in range(5):
        E, _, iters, resid, _ = plan.solve(kb[p], kk[p], pol[p, 0::2] + 1j * pol[p, 1::2], tol=1e-12)
        assert iters == it[p] and resid == res[p] and torch.equal(E, F[p])
    plan.close()


def test_cluster_gram_schmidt_at_32_cubed():
    """32^3 orders (98 304 complex numbers per vector = 6144 per CTA of a 16-CTA cluster) is the largest vector the cluster
    Gram-Schmidt kernel holds on chip; it agrees with the two-sweep kernels and the field satisfies the equation at
    sampled harmonics (the oracle's O(n) row sums)."""
    from test_gpu_solve import _check_equation_rows
    geo = wl.sphere_lattice((32, 32, 32))
    kb, pol = np.array([0.0, 0.0, 1.2 * TWO_PI]), np.array([1.0, 0.0, 0.0], dtype=complex)
    plan = gsm.plan_from_geometry(geo, max_iters=80)
    E, hist, iters, resid, st = plan.solve(kb, TWO_PI, pol, tol=1e-12)
    prof = plan.profile_read()
    assert st == gsm.OK and resid <= 1e-10 and prof["arnoldi_mgs"][0] >= iters and prof["sweep_dots"][0] == 0
    plan.close()
    two = gsm.plan_from_geometry(geo, max_iters=80, flags=gsm.FLAG_TWO_SWEEP)
    E2, _, it2, res2, st2 = two.solve(kb, TWO_PI, pol, tol=1e-12)
    assert st2 == gsm.OK and abs(it2 - iters) <= 1 and rel(E.cpu().numpy(), E2.cpu().numpy()) <= 1e-10
    two.close()
    _check_equation_rows(geo, coeffs(geo), E.cpu().numpy()[None], kb[None], np.array([TWO_PI]), pol[None], 6)


def test_group_concurrent_iteration_is_bit_identical():
    """A lock-step batch of 8 or more solves iterates as 2-4 groups on streams of their own (one group's Gram-Schmidt beside
    another's apply); with per-launch profiling on it runs as one group.  Same kernels and reductions per solve: results
    are identical bit for bit, for mixed convergence, a zero source, guesses, and a batch that stops at max_iters."""
    geo = wl.sphere_lattice((17, 17, 17))
    npts = 26
    kb, kk, pol = wl.scan_points(wl.kappa_mesh(1.02, 1.30, npts), 2, 0)
    kb[5] = [0.3, -0.2, 1.15 * TWO_PI]
    pol[9] = 0.0
    plan = gsm.plan_from_geometry(geo, max_iters=80, max_batch=npts)
    Fa = torch.empty((npts, 3, 17, 17, 17), dtype=torch.complex128, device="cuda")
    Fb = torch.zeros_like(Fa)
    ra, ia, resa, sta = plan.scan(kb, kk, pol, tol=1e-12, fields=Fa)                 # 4 groups
    plan.profile(True)
    rb, ib, resb, stb = plan.scan(kb, kk, pol, tol=1e-12, fields=Fb)                 # one group
    plan.profile(False)
    assert sta == stb == gsm.OK and len(set(ia.tolist())) > 2 and ia[9] == 0
    assert np.array_equal(ia, ib) and np.array_equal(ra, rb) and np.array_equal(resa, resb) and torch.equal(Fa, Fb)
    assert np.all(resa <= 1e-10)
    # from guesses (the fields just computed, perturbed): the groups share the apply that forms r0
    X0 = Fa * (1.0 + 1e-4)
    Fc, Fd = torch.empty_like(Fa), torch.empty_like(Fa)
    rc, ic, resc, _ = plan.scan(kb, kk, pol, tol=1e-12, x0=X0, fields=Fc)
    plan.profile(True)
    rd, idd, resd, _ = plan.scan(kb, kk, pol, tol=1e-12, x0=X0, fields=Fd)
    plan.profile(False)
    assert np.array_equal(ic, idd) and np.array_equal(rc, rd) and torch.equal(Fc, Fd) and ic.max() < ia.max()
    plan.close()
    short = gsm.plan_from_geometry(geo, max_iters=6, max_batch=npts)
    r1, i1, s1, st1 = short.scan(kb, kk, pol, tol=1e-12)
    short.profile(True)
    r2, i2, s2, st2 = short.scan(kb, kk, pol, tol=1e-12)
    assert st1 == st2 == gsm.NOT_CONVERGED and np.array_equal(i1, i2) and np.array_equal(r1, r2) and np.array_equal(s1, s2)
    assert np.all(np.delete(i1, 9) == 6)
    short.close()


def test_tetragonal_lattice_normal_surface_and_period_sweep_vs_oracle_goldens():
    """SURVEY 8(f) #4, the rest of the row (Fig. 4): spherical air cavities (R = 0.02 lambda) in n = 1.5 on
    a simple tetragonal lattice at the constant filling factor 0.155.  (1) Lambda_x / Lambda_y,z = 0.7 and 1.3: BOTH sheets
    of the Fresnel normal surface along 4 seeded directions of the xz plane - amplitude y (ordinary) and y x s
    (extraordinary), response = projection on the amplitude (reading R28) - 8 lines per call of gsm_retrieve_neff_many,
    against the oracle's dense-LU retrieval (tests/golden/oracle_neff.txt, group `tetra`).  (2) Five ratios at constant
    filling through gsm_plan_set_cell, k || z with a = x and a = y, against the same goldens and the Maxwell-Garnett line."""
    gold = load_oracle_golden()
    mg = load_golden()["n_mg_uniaxial"]
    dirs, pols = wl.normal_surface_lines(4)
    plan = gsm.plan_from_geometry(wl.tetragonal_cavities(0.7), max_iters=100, max_batch=8 * 29)
    for ratio in (0.7, 1.3):
        geo = wl.tetragonal_cavities(ratio)
        plan.set_cell(geo.periods, shapes=geo.shapes, eps_bg=geo.eps_bg, eps_b=geo.eps_b)
        n, eps, zeta, ls, st = plan.retrieve_neff_many(dirs, pols.astype(complex), -1, TWO_PI, 1.39, 1.46, tol=1e-12)
        assert st == gsm.OK and np.all(ls == gsm.OK)
        for i in range(8):
            key = f"tetra_{ratio:g}_surf_{i}"
            assert abs(n[i].real - gold[key + "_neff_re"]) <= 1e-8 and abs(n[i].imag) <= 1e-9, key
            assert abs(eps[i].real - gold[key + "_eps_re"]) <= 1e-8
            zo = complex(gold[key + "_zeta_re"], gold[key + "_zeta_im"])
            assert abs(zeta[i] - zo) <= 1e-6 * abs(zo)
        # uniaxial crystal, axis x: the ordinary sheet is (nearly) a circle, the extraordinary one is not, and the two
        # approach each other as s turns towards the axis (rows are sorted by the angle between s and z)
        no, ne = n[0::2].real, n[1::2].real
        assert np.ptp(no) <= 5e-5 and np.ptp(ne) >= 1e-3
        assert np.all(np.diff(np.abs(ne - no)) < 0)
        assert (ne[0] > no[0]) == (ratio < 1.0)
    zdir = np.array([[0.0, 0.0, 1.0], [0.0, 0.0, 1.0]])
    xy = np.array([[1.0, 0, 0], [0, 1.0, 0]], dtype=complex)
    nx, ny = [], []
    for ratio in (0.7, 0.85, 1.0, 1.15, 1.3):
        geo = wl.tetragonal_cavities(ratio)
        plan.set_cell(geo.periods, shapes=geo.shapes, eps_bg=geo.eps_bg, eps_b=geo.eps_b)
        n, eps, zeta, ls, st = plan.retrieve_neff_many(zdir, xy, -1, TWO_PI, 1.39, 1.46, tol=1e-12)
        assert st == gsm.OK and np.all(ls == gsm.OK)
        for i, nm in enumerate(("ax", "ay")):
            assert abs(n[i].real - gold[f"tetra_{ratio:g}_kz_{nm}_neff_re"]) <= 1e-8
        nx.append(n[0].real); ny.append(n[1].real)
    nx, ny = np.array(nx), np.array(ny)
    assert abs(nx[2] - ny[2]) <= 1e-10                         # equal periods: isotropic
    assert 0.0 < nx[2] - mg < 3e-3                             # finite periods raise the index above Maxwell-Garnett
    assert np.all(np.diff(nx) < 0) and np.all(np.diff(ny) > 0)  # extraordinary falls, ordinary rises with Lambda_x / Lambda_y,z
    assert nx[-1] < mg                                         # "one of the effective indices ... can become lower than" the MG value
    plan.close()
