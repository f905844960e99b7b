"""GPU parity of the GMRES solve, the batched scan and the pole search against the CPU oracle (dense LU where the
oracle can afford it, the oracle's own full GMRES above that).

Bars (BASELINE.json north_star): relative L2 field error <= 1e-9, true Krylov residual <= 1e-10, retrieved
eps_eff within 1e-8.  Solves run to tol 1e-12 (reading R10: field error <= cond(A) x residual).
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

from conftest import load_oracle_golden  # noqa: E402
from oracle import gsm_oracle as orc  # noqa: E402
from paper_1501_01752_b200 import gsm, workloads as wl  # noqa: E402

TWO_PI = 2.0 * np.pi


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def coeffs(geo):
    if geo.voxels is not None:
        return orc.coeffs_voxel(geo.voxels, geo.orders, geo.eps_b)
    return orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)


def test_config1_sphere_7cubed_vs_dense_lu():
    """BASELINE config 1: 7^3 orders, eps 4 sphere R = 0.3 Lambda, Lambda = 0.2 lambda, k along z, a = x."""
    geo = wl.sphere_lattice((7, 7, 7))
    plan = gsm.plan_from_geometry(geo, max_iters=64)
    kb, k0, pol = np.array([0.0, 0.0, 1.2 * TWO_PI]), TWO_PI, np.array([1.0, 0.0, 0.0], dtype=complex)
    E, hist, iters, resid, st = plan.solve(kb, k0, pol, tol=1e-12)
    ref = orc.solve_dense(coeffs(geo), geo.periods, geo.orders, kb, k0, geo.eps_b, pol)
    assert st == gsm.OK
    assert resid <= 1e-10
    assert rel(E.cpu().numpy(), ref) <= 1e-9
    # history: non-increasing, last entry below tol, length in the paper's band (~10 .. ~50)
    assert len(hist) == iters and np.all(np.diff(hist) <= 1e-15) and hist[-1] <= 1e-12
    _, ohist, oiters = orc.solve_gmres(coeffs(geo), geo.periods, geo.orders, kb, k0, geo.eps_b, pol, tol=1e-12)
    assert abs(iters - oiters) <= 2
    assert 5 <= iters <= 60
    # lossless centred cell, real kappa: the solution is real (SURVEY 8(c) invariants)
    assert np.max(np.abs(E.cpu().numpy().imag)) <= 1e-12
    plan.close()


def test_homogeneous_cell_lucky_breakdown():
    """Delta eps = 0: A = I, E = E_inc after one iteration with h_21 = 0 (reading R23)."""
    geo = wl.sphere_lattice((5, 5, 5), eps=1.0)
    plan = gsm.plan_from_geometry(geo)
    pol = np.array([0.3 - 0.2j, 1.0, 0.5j])
    E, hist, iters, resid, st = plan.solve([0.1, 0.2, 1.1 * TWO_PI], TWO_PI, pol, tol=1e-10)
    assert st == gsm.OK and iters == 1 and resid <= 1e-15
    ref = orc.incident(geo.orders, pol)
    assert np.max(np.abs(E.cpu().numpy() - ref)) <= 1e-15
    plan.close()


def test_guessed_start_near_breakdown_stays_finite():
    """Reading R23 with a guessed start (oracle pin: test_gmres_guess_off_by_one_eigenvector_...): x0 = x* + 1e-7 u with u
    an eigenvector of A, and a tolerance that cannot be met.  After one iteration nothing but rounding is left of A v_0;
    whether the device calls that a breakdown (h_10 <= eps ||A v_0||) or keeps orthogonalising rounding noise, the
    returned field must be the exact solution, finite, with a true residual at rounding level."""
    geo = wl.Geometry("uniform", (0.2, 0.2, 0.2), (3, 3, 3),
                      [dict(kind=wl.BOX, center=(0, 0, 0), size=(0.2, 0.2, 0.2), eps=2.5)], 1.0, 1.0, None, ())
    c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
    kb = np.array([[0.0, 0.0, 1.3 * TWO_PI]])
    ref = orc.solve_dense(c, geo.periods, geo.orders, kb[0], TWO_PI, geo.eps_b, [1.0, 0, 0])
    u = np.zeros_like(ref)
    u[1, 2, 1, 1] = 1.0
    plan = gsm.plan_from_geometry(geo, max_iters=20)
    fields = torch.empty((1, 3, 3, 3, 3), dtype=torch.complex128, device="cuda")
    x0 = torch.from_numpy((ref + 1e-7 * u)[None]).cuda()
    resp, iters, resid, st = plan.scan(kb, [TWO_PI], np.array([[1.0, 0, 0, 0, 0, 0]]), tol=1e-30, fields=fields, x0=x0)
    E = fields.cpu().numpy()[0]
    assert st in (gsm.OK, gsm.NOT_CONVERGED) and 1 <= iters[0] <= 20
    assert np.all(np.isfinite(E.view(np.float64))) and np.isfinite(resid[0]) and resid[0] <= 1e-14
    assert np.linalg.norm(E - ref) / np.linalg.norm(ref) <= 1e-13
    plan.close()


def test_uniform_cell_closed_form():
    """c_d = Delta delta_d0: E_0 = a (kappa^2 - k0^2 eps_b)/(kappa^2 - k0^2 eps_2) for transverse a."""
    eps2, eps_b = 2.5, 1.0
    geo = wl.Geometry("uniform", (0.2, 0.2, 0.2), (3, 3, 3),
                      [dict(kind=wl.BOX, center=(0, 0, 0), size=(0.2, 0.2, 0.2), eps=eps2)], 1.0, eps_b, None, ())
    plan = gsm.plan_from_geometry(geo)
    kappa, k0 = 1.3 * TWO_PI, TWO_PI
    E, _, _, resid, _ = plan.solve([0, 0, kappa], k0, [1.0, 0, 0], tol=1e-13)
    e0 = orc.zero_order(E.cpu().numpy())
    assert abs(e0[0] - (kappa**2 - k0**2 * eps_b) / (kappa**2 - k0**2 * eps2)) <= 1e-12
    E, _, _, _, _ = plan.solve([0, 0, kappa], k0, [0, 0, 1.0], tol=1e-13)      # longitudinal: a eps_b / eps_2
    assert abs(orc.zero_order(E.cpu().numpy())[2] - eps_b / eps2) <= 1e-12
    plan.close()


def test_max_iters_reports_not_converged():
    geo = wl.sphere_lattice((7, 7, 7))
    plan = gsm.plan_from_geometry(geo, max_iters=4)
    E, hist, iters, resid, st = plan.solve([0, 0, 1.2 * TWO_PI], TWO_PI, [1.0, 0, 0], tol=1e-12)
    assert st == gsm.NOT_CONVERGED and iters == 4 and len(hist) == 4
    assert abs(resid - hist[-1]) <= 1e-10          # best iterate is returned: true residual = estimate
    plan.close()


def test_complex_eps_b_and_offcentre_shapes_vs_dense_lu():
    shapes = [dict(kind=wl.ELLIPSOID, center=(0.03, -0.02, 0.05), size=(0.06, 0.05, 0.04), eps=8.0 + 0.5j),
              dict(kind=wl.BOX, center=(-0.05, 0.04, 0.0), size=(0.05, 0.08, 0.3), eps=2.5)]
    geo = wl.Geometry("lossy", (0.2, 0.25, 0.3), (5, 4, 6), shapes, 1.5, 1.3 + 0.1j, None, ())
    plan = gsm.plan_from_geometry(geo, max_iters=100)
    kb, k0, pol = np.array([0.4, -0.3, 1.4 * TWO_PI]), 0.9 * TWO_PI, np.array([1.0, 0.5j, -0.2])
    E, hist, iters, resid, st = plan.solve(kb, k0, pol, tol=1e-12)
    ref = orc.solve_dense(coeffs(geo), geo.periods, geo.orders, kb, k0, geo.eps_b, pol)
    assert st == gsm.OK and resid <= 1e-10 and rel(E.cpu().numpy(), ref) <= 1e-9
    plan.close()


def test_config2_laminate_scan_vs_dense_lu_and_rytov_pole():
    """BASELINE config 2 (1x1x63): batched scan in chunks (npts > max_batch), TE along z; pole vs oracle pole search."""
    geo = wl.laminate((1, 1, 63))
    plan = gsm.plan_from_geometry(geo, max_iters=80, max_batch=8)
    c = coeffs(geo)
    k0 = TWO_PI * 0.25 * 20 / 64                      # Lambda_z / lambda = 0.078 (pass band, reading R21)
    # Rytov TE dispersion root (closed form) brackets the mesh
    d1 = d2 = 0.5
    k1, k2 = k0 * 1.0, k0 * 3.0
    cosK = np.cos(k1 * d1) * np.cos(k2 * d2) - 0.5 * (k1 / k2 + k2 / k1) * np.sin(k1 * d1) * np.sin(k2 * d2)
    K_rytov = np.arccos(cosK)
    npts = 19
    step = 0.01 * K_rytov
    kappa = K_rytov + step * (np.arange(npts) - (npts - 1) / 2 + 0.5)      # pole mid-way between nodes (R16)
    kb, kk, pol = wl.scan_points(kappa, 2, 0, k0)
    fields = torch.empty((npts, 3, 1, 1, 63), dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, kk, pol, tol=1e-12, fields=fields)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    xi_ref = np.zeros(npts, dtype=complex)
    F = fields.cpu().numpy()
    for p in range(npts):
        ref = orc.solve_dense(c, geo.periods, geo.orders, kb[p], k0, geo.eps_b, [1.0, 0, 0])
        xi_ref[p] = orc.zero_order(ref)[0]
        # near-pole points are compared through xi and eta (reading R10); fields where cond is moderate
        if abs(kappa[p] - K_rytov) > 3 * step:
            assert rel(F[p], ref) <= 1e-9
    assert np.max(np.abs(resp[:, 0] - xi_ref) / np.abs(xi_ref)) <= 1e-8
    eta, zeta, best = gsm.pole_search(kappa, resp[:, 0], 5, 10)
    eta_o, zeta_o = orc.pole_search(kappa, xi_ref, 5, 10)
    bo = orc.select_pole(eta_o, zeta_o, kappa[0], kappa[-1])
    assert best >= 0 and bo >= 0
    n_gpu, eps_gpu = eta[best] / k0, (eta[best] / k0) ** 2
    n_orc, eps_orc = orc.retrieve_eps(eta_o[bo], k0)
    assert abs(eps_gpu - eps_orc) <= 1e-8
    assert abs(zeta[best] - zeta_o[bo]) <= 1e-7 * abs(zeta_o[bo])
    assert abs(eta[best].real - K_rytov) <= 1e-6 * K_rytov      # truncation error ~N^-3
    plan.close()


def test_config3_ellipsoid_15cubed_vs_oracle_gmres():
    """BASELINE config 3 at one (k, omega) point per tensor entry: oracle = its own full GMRES on the O(n^2) product."""
    geo = wl.ellipsoid_lattice((15, 15, 15))
    plan = gsm.plan_from_geometry(geo, max_iters=80, max_batch=3)
    c = coeffs(geo)
    pts = [(2, 0, 1.20), (0, 1, 1.18), (1, 2, 1.15)]          # (prop axis, pol axis, n_i): reading R14
    kb = np.zeros((3, 3)); pol = np.zeros((3, 3), dtype=complex)
    for i, (pa, qa, ni) in enumerate(pts):
        kb[i, pa] = ni * TWO_PI
        pol[i, qa] = 1.0
    fields = torch.empty((3, 3, 15, 15, 15), dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, np.full(3, TWO_PI), pol, tol=1e-12, fields=fields)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    F = fields.cpu().numpy()
    for i in range(3):
        ref, ohist, oit = orc.solve_gmres(c, geo.periods, geo.orders, kb[i], TWO_PI, geo.eps_b, pol[i], tol=1e-13,
                                          max_iters=120, matvec=orc.toeplitz_matvec_c)
        assert rel(F[i], ref) <= 1e-9
        assert abs(int(iters[i]) - oit) <= 4
        assert abs(resp[i, pts[i][1]] - orc.zero_order(ref)[pts[i][1]]) <= 1e-9 * abs(orc.zero_order(ref)[pts[i][1]])
    plan.close()


def test_scan_mixed_convergence_and_repeatability():
    """Solves of one lock-step batch stop at different iterations; results do not depend on the batch grouping."""
    geo = wl.sphere_lattice((7, 7, 7))
    kappa = wl.kappa_mesh(1.02, 1.30, 12)
    kb, kk, pol = wl.scan_points(kappa, 2, 0)
    pa = gsm.plan_from_geometry(geo, max_batch=12)
    pb = gsm.plan_from_geometry(geo, max_batch=5)
    ra, ia, _, _ = pa.scan(kb, kk, pol, tol=1e-11)
    rb, ib, _, _ = pb.scan(kb, kk, pol, tol=1e-11)
    assert len(set(ia.tolist())) > 1
    assert np.array_equal(ia, ib) and np.array_equal(ra, rb)      # deterministic reductions: bit-identical
    # residual history of every solve of the batch (gsm_plan_history), against gsm_solve's own history of that point
    for b in (0, 5, 11):
        h = pa.history(b)
        _, hs, its, _, _ = pb.solve(kb[b], kk[b], pol[b, 0::2] + 1j * pol[b, 1::2], tol=1e-11)
        assert len(h) == ia[b] == its and np.array_equal(h, hs) and h[-1] <= 1e-11 < h[-2]
    with pytest.raises(gsm.GsmError):
        pa.history(12)
    pa.close(); pb.close()


def test_config5a_bench_configuration_sampled_points():
    """BASELINE config 5a exactly as bench.py times it (voxel composite, 31^3 orders, 256 points, the 64-point fast path
    and the cluster MGS kernel), both as one lock-step batch from a zero start (gsm_scan) and as the 5-wave mesh scan with
    interpolated guesses that bench.py's headline uses (gsm_scan_mesh): every solve meets the residual bar; sampled points
    (one per wave of the mesh scan) are compared field by field with the oracle's own GMRES on the O(n^2) product."""
    geo = wl.voxel_composite((31, 31, 31), nv=128)
    kappa = wl.kappa_mesh(1.05, 1.20, 256)
    kb, kk, pol = wl.scan_points(kappa, 2, 0)
    plan = gsm.plan_from_geometry(geo, max_iters=64, max_batch=256)
    fields = torch.empty((256, 3, 31, 31, 31), dtype=torch.complex128, device="cuda")
    c = coeffs(geo)
    refs = {p: orc.solve_gmres(c, geo.periods, geo.orders, kb[p], TWO_PI, geo.eps_b, [1.0, 0, 0], tol=1e-13,
                               max_iters=100, matvec=orc.toeplitz_matvec_c) for p in (2, 3, 4, 8, 201)}
    totals = []
    for levels in (None, 5):
        resp, iters, resid, st = plan.scan(kb, kk, pol, tol=1e-12, fields=fields, levels=levels)
        assert st == gsm.OK and np.all(resid <= 1e-10)
        assert iters.max() <= 64 and (levels or iters.min() >= 10)      # PAPER.md:103 band (zero start)
        for p, (ref, _, oit) in refs.items():     # mesh scan: 8 is solved in wave 1 (guessed from wave 0), the others in the waves after it
            assert rel(fields[p].cpu().numpy(), ref) <= 1e-9
            assert levels or abs(int(iters[p]) - oit) <= 5
            assert abs(resp[p, 0] - orc.zero_order(ref)[0]) <= 1e-9 * abs(orc.zero_order(ref)[0])
        # the response is the m = 0 entry of the returned field, for every point
        F0 = fields[:, :, 15, 15, 15].cpu().numpy()
        assert np.array_equal(F0, resp)
        totals.append(int(iters.sum()))
    assert totals[1] < 0.5 * totals[0]            # the guesses save iterations (measured at 1e-10: 40.8 -> 8.2 per solve)
    plan.close()


def test_config3_eps_xx_retrieval_vs_oracle_pipeline():
    """BASELINE config 3, tensor entry xx (k || z, a = x, reading R14): scan -> pole search -> eps_eff on both sides.
    The kappa mesh is placed by the ORACLE's coarse scan (pole mid-way between two nodes, reading R16)."""
    geo = wl.ellipsoid_lattice((15, 15, 15))
    c = coeffs(geo)
    k0 = TWO_PI

    def oracle_xi(kap):
        out = np.zeros(len(kap), dtype=complex)
        for i, kv in enumerate(kap):
            E, _, _ = orc.solve_gmres(c, geo.periods, geo.orders, np.array([0, 0, kv]), k0, geo.eps_b, [1.0, 0, 0],
                                      tol=1e-13, max_iters=150, matvec=orc.toeplitz_matvec_c)
            out[i] = orc.zero_order(E)[0]
        return out
    coarse = wl.kappa_mesh(1.02, 1.30, 29)
    xc = oracle_xi(coarse)
    eta_c, zeta_c = orc.pole_search(coarse, xc, 5, 10)
    bc = orc.select_pole(eta_c, zeta_c, coarse[0], coarse[-1])
    assert bc >= 0
    step = 0.002 * k0
    fine = eta_c[bc].real + step * (np.arange(18) - 8.5)          # estimate falls mid-way between two nodes
    xi_o = oracle_xi(fine)
    eta_o, zeta_o = orc.pole_search(fine, xi_o, 5, 10)
    bo = orc.select_pole(eta_o, zeta_o, fine[0], fine[-1])
    n_o, eps_o = orc.retrieve_eps(eta_o[bo], k0)

    plan = gsm.plan_from_geometry(geo, max_iters=120, max_batch=18)
    kb, kk, pol = wl.scan_points(fine, 2, 0)
    resp, iters, resid, st = plan.scan(kb, kk, pol, tol=1e-12)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    eta, zeta, best = gsm.pole_search(fine, resp[:, 0], 5, 10)
    assert best >= 0
    eps_g = (eta[best] / k0) ** 2
    assert abs(eps_g - eps_o) <= 1e-8
    assert abs(eps_g.real - load_oracle_golden()["cfg3_15_xx_eps_re"]) <= 1e-8      # oracle-written golden (two-stage)
    plan.close()


def test_degenerate_inputs_empty_scan_zero_source_and_largest_orders():
    geo = wl.sphere_lattice((5, 5, 5))
    plan = gsm.plan_from_geometry(geo, max_batch=4)
    resp, iters, resid, st = plan.scan(np.zeros((0, 3)), np.zeros(0), np.zeros((0, 6)), tol=1e-10)
    assert st == gsm.OK and resp.shape == (0, 3) and len(iters) == 0
    # zero source: b = 0 -> E = 0 without iterating; mixed with a normal point in the same batch
    kb = np.array([[0, 0, 1.2 * TWO_PI], [0, 0, 1.2 * TWO_PI]])
    pol = np.zeros((2, 6)); pol[1, 0] = 1.0
    fields = torch.full((2, 3, 5, 5, 5), 7.0, dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, np.full(2, TWO_PI), pol, tol=1e-11, fields=fields)
    assert st == gsm.OK and iters[0] == 0 and iters[1] > 3 and resid[0] == 0.0 and resid[1] <= 1e-10
    assert float(fields[0].abs().max()) == 0.0 and np.all(resp[0] == 0)
    plan.close()
    # largest supported order count per axis (256 -> 512-point axis) is accepted; 257 is rejected; so is max_iters > cap
    big = wl.Geometry("max", (0.2, 0.2, 0.2), (256, 1, 2), geo.shapes, 1.0, 1.0, None, ())
    p2 = gsm.plan_from_geometry(big)
    assert p2.info()["fft_grid"] == (512, 1, 4)
    p2.close()
    with pytest.raises(gsm.GsmError) as e:
        gsm.Plan((0.2, 0.2, 0.2), (257, 1, 1), shapes=geo.shapes)
    assert e.value.status == gsm.E_INVALID
    with pytest.raises(gsm.GsmError) as e:
        gsm.Plan((0.2, 0.2, 0.2), (5, 5, 5), shapes=geo.shapes, max_iters=gsm.MAX_ITERS + 1)
    assert e.value.status == gsm.E_INVALID


def test_config2_laminate_in_plane_te_tm_vs_dense_lu():
    """BASELINE config 2, propagation along x (in the layer planes): a = y (TE) and a = z (TM), fields vs dense LU."""
    geo = wl.laminate((1, 1, 63))
    plan = gsm.plan_from_geometry(geo, max_iters=120, max_batch=6)
    c = coeffs(geo)
    k0 = TWO_PI * 0.25 * 24 / 64
    kb = np.zeros((6, 3)); pol = np.zeros((6, 3), dtype=complex)
    ns = [1.9, 2.1, 2.3, 1.2, 1.3, 1.45]                  # TE points around n ~ sqrt(5), TM points around n ~ sqrt(1.8)
    for i, n in enumerate(ns):
        kb[i, 0] = n * k0
        pol[i, 1 if i < 3 else 2] = 1.0
    fields = torch.empty((6, 3, 1, 1, 63), dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, np.full(6, k0), pol, tol=1e-12, fields=fields)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    F = fields.cpu().numpy()
    for i in range(6):
        ref = orc.solve_dense(c, geo.periods, geo.orders, kb[i], k0, geo.eps_b, pol[i])
        assert rel(F[i], ref) <= 1e-9
    plan.close()


def test_config4_woodpile_31cubed_three_directions():
    """BASELINE config 4: one (k, omega) point per search direction (z,x), (x,y), (x,z) in one batch.  The (z,x) solve is
    compared with the oracle's GMRES; all three are checked against the equation itself at sampled harmonics with the
    oracle's O(n) row sums (A E = b)."""
    geo = wl.woodpile((31, 31, 31))
    plan = gsm.plan_from_geometry(geo, max_iters=100, max_batch=3)
    c = coeffs(geo)
    pts = [(2, 0, 1.35), (0, 1, 1.36), (0, 2, 1.27)]
    kb = np.zeros((3, 3)); pol = np.zeros((3, 3), dtype=complex)
    for i, (pa, qa, ni) in enumerate(pts):
        kb[i, pa] = ni * TWO_PI
        pol[i, qa] = 1.0
    fields = torch.empty((3, 3, 31, 31, 31), dtype=torch.complex128, device="cuda")
    resp, iters, resid, st = plan.scan(kb, np.full(3, TWO_PI), pol, tol=1e-12, fields=fields)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    F = fields.cpu().numpy()
    ref, _, oit = orc.solve_gmres(c, geo.periods, geo.orders, kb[0], TWO_PI, geo.eps_b, pol[0], tol=1e-13, max_iters=150,
                                  matvec=orc.toeplitz_matvec_c)
    assert rel(F[0], ref) <= 1e-9 and abs(int(iters[0]) - oit) <= 5
    _check_equation_rows(geo, c, F, kb, np.full(3, TWO_PI), pol, 10)
    plan.close()


def _check_equation_rows(geo, c, F, kb, k0, pol, nsamp):
    """(A E)_m = b_m at sampled harmonics, A E evaluated by the oracle's row sum (no FFT, O(n) per row)."""
    rng = np.random.default_rng(17)
    N = geo.orders
    i0 = tuple(n // 2 for n in N)             # index of m = 0 (reading R1: odd N: (N-1)/2, even N: N/2)
    for b in range(F.shape[0]):
        k = orc.wavevectors(geo.periods, N, kb[b])
        kb2 = k0[b] ** 2 * geo.eps_b
        scale = np.abs(F[b]).max()
        for s in [i0, (0, 0, 0)] + [tuple(int(rng.integers(0, N[a])) for a in range(3)) for _ in range(nsamp)]:
            T = orc.toeplitz_row(c, F[b], s)
            km = k[(slice(None),) + s]
            lhs = F[b][(slice(None),) + s] - (kb2 * T - km * np.dot(km, T)) / (np.dot(km, km) - kb2)
            rhs = pol[b] if s == i0 else np.zeros(3)
            assert np.max(np.abs(lhs - rhs)) <= 1e-9 * max(1.0, scale)


def test_config5b_63cubed_single_solve_vs_oracle_solution():
    """BASELINE config 5b at the north_star's tolerance: one solve at 63^3 orders against the ORACLE'S OWN SOLUTION of the same
    point (full GMRES to 1e-13 with the O(n^2) Toeplitz product, ~45 minutes of host time, stored once by
    tests/golden/make_oracle_goldens.py --only cfg5b): the 0-th order response, the norm of the field and 4096 seeded
    entries of it.  Field entries within 1e-9 of the field's rms entry, sampled relative L2 error, xi and norm within 1e-9."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_cfg5b_63.txt")
    if not os.path.exists(path):
        pytest.skip("tests/golden/oracle_cfg5b_63.txt has not been generated (make_oracle_goldens.py --only cfg5b)")
    head, idx, val = {}, [], []
    with open(path) as f:
        for line in f:
            t = line.split("#")[0].split()
            if not t:
                continue
            if t[0] == "sample":
                idx.append(int(t[1])); val.append(complex(float(t[2]), float(t[3])))
            else:
                head[t[0]] = float(t[1].replace("np.float64(", "").rstrip(")"))   # numpy 2 prints its scalars as np.float64(..)
    idx, val = np.array(idx), np.array(val)
    assert len(idx) == 4096 and head["true_rel_resid"] <= 1e-11 and head["estimated_rel_resid"] <= 1e-13
    geo = wl.voxel_composite((63, 63, 63), nv=128)
    plan = gsm.plan_from_geometry(geo, max_iters=100, max_batch=1)
    kb = np.array([0.0, 0.0, 1.12 * TWO_PI]); pol = np.array([1.0, 0, 0], dtype=complex)
    E, hist, iters, resid, st = plan.solve(kb, TWO_PI, pol, tol=1e-13)          # the oracle's own tolerance
    assert st == gsm.OK and resid <= 1e-10 and abs(iters - int(head["iters"])) <= 8
    F = E.cpu().numpy()
    n3 = F.size
    rms = head["norm_E"] / np.sqrt(n3)
    got = F.ravel()[idx]
    assert np.max(np.abs(got - val)) <= 1e-9 * rms
    assert np.linalg.norm(got - val) / np.linalg.norm(val) <= 1e-9
    assert abs(np.linalg.norm(F) - head["norm_E"]) <= 1e-9 * head["norm_E"]
    xi = orc.zero_order(F)
    xo = np.array([complex(head[f"xi{a}_re"], head[f"xi{a}_im"]) for a in range(3)])
    assert np.max(np.abs(xi - xo)) <= 1e-9 * np.max(np.abs(xo))
    plan.close()


def test_config5b_63cubed_single_solve_satisfies_the_equation():
    """BASELINE config 5b: one solve at 63^3 orders (128-point xy fast path, generic z passes, two-sweep Gram-Schmidt).
    The oracle cannot afford a solve at this size; the returned field is checked against the equation at sampled
    harmonics through the oracle's row sums, and against the solver's own true residual."""
    geo = wl.voxel_composite((63, 63, 63), nv=128)
    plan = gsm.plan_from_geometry(geo, max_iters=80, max_batch=1)
    kb = np.array([0.0, 0.0, 1.12 * TWO_PI]); pol = np.array([1.0, 0, 0], dtype=complex)
    E, hist, iters, resid, st = plan.solve(kb, TWO_PI, pol, tol=1e-12)
    assert st == gsm.OK and resid <= 1e-10 and 20 <= iters <= 70 and np.all(np.diff(hist) <= 1e-15)
    c = coeffs(geo)
    _check_equation_rows(geo, c, E.cpu().numpy()[None], kb[None], np.array([TWO_PI]), pol[None], 8)
    plan.close()


@pytest.mark.parametrize("N", [128, 256])
def test_table1_large_orders_single_solve_satisfies_the_equation(N):
    """128^3 and 256^3 orders (Table 1's last two columns: 6.3 M / 50 M unknowns, 256^3 / 512^3 FFT
    grid) as ONE solve on the device: split plane pass, generic z passes, two-sweep Gram-Schmidt.  At 256^3 the paper's
    GMRES vectors did not fit its 6 GB card and were streamed from host RAM; here the whole basis
    (41 x 805 MB) stays in HBM.  The
    workload has the shape the paper states (lattice of spheres with refractive index 3 in air, GMRES to 1e-8, "about 30
    iterations"); radius, period and wavevector are not printed (here R = 0.3 Lambda, Lambda = 0.3 lambda,
    k = 1.3 k0 z).  The oracle cannot afford a solve at this size: the field is checked against the equation at sampled
    harmonics through the oracle's O(n) row sums, and against the solver's own true residual."""
    geo = wl.sphere_lattice((N, N, N), period=0.3, radius_frac=0.3, eps=9.0)
    plan = gsm.plan_from_geometry(geo, max_iters=40, max_batch=1)
    assert plan.info()["fft_grid"] == (2 * N, 2 * N, 2 * N)
    kb = np.array([0.0, 0.0, 1.3 * TWO_PI]); pol = np.array([1.0, 0, 0], dtype=complex)
    E, hist, iters, resid, st = plan.solve(kb, TWO_PI, pol, tol=1e-10)
    assert st == gsm.OK and resid <= 1e-9 and 20 <= iters <= 40 and np.all(np.diff(hist) <= 1e-15)
    F = E.cpu().numpy()[None]
    plan.close()
    del E
    torch.cuda.empty_cache()
    c = coeffs(geo)
    rng = np.random.default_rng(17)
    i0 = (N // 2, N // 2, N // 2)          # even order count: m = 0 sits at index N/2 (reading R1)
    k = orc.wavevectors(geo.periods, geo.orders, kb)
    kb2 = TWO_PI ** 2 * geo.eps_b
    scale = np.abs(F[0]).max()
    for s in [i0, (0, 0, 0), (N - 1, N - 1, N - 1)] + [tuple(int(rng.integers(0, N)) for _ in range(3)) for _ in range(5)]:
        T = orc.toeplitz_row(c, F[0], s)
        km = k[(slice(None),) + s]
        lhs = F[0][(slice(None),) + s] - (kb2 * T - km * np.dot(km, T)) / (np.dot(km, km) - kb2)
        rhs = pol if s == i0 else np.zeros(3)
        assert np.max(np.abs(lhs - rhs)) <= 1e-8 * max(1.0, scale)


def test_plans_of_different_sizes_coexist():
    """Kernel attributes (dynamic shared memory, cluster size) are per function: a small plan created after a large one
    must not shrink what the large one needs, and vice versa."""
    big = gsm.plan_from_geometry(wl.woodpile((31, 31, 31)), max_iters=40, max_batch=2)
    small = gsm.plan_from_geometry(wl.sphere_lattice((7, 7, 7)), max_iters=40, max_batch=2)
    kb = np.array([[0, 0, 1.35 * TWO_PI], [0, 0, 1.3 * TWO_PI]]); pol = np.zeros((2, 6)); pol[:, 0] = 1.0
    r1, it1, res1, st1 = big.scan(kb, np.full(2, TWO_PI), pol, tol=1e-8)
    r2, it2, res2, st2 = small.scan(kb, np.full(2, TWO_PI), pol, tol=1e-8)
    r3, it3, res3, st3 = big.scan(kb, np.full(2, TWO_PI), pol, tol=1e-8)
    assert st1 == st2 == st3 == gsm.OK and np.all(res1 <= 1e-7) and np.all(res2 <= 1e-7)
    assert np.array_equal(r1, r3) and np.array_equal(it1, it3)
    big.close(); small.close()


def test_retrieve_neff_config1_vs_oracle():
    """gsm_retrieve_neff (two-stage scan + pole search, reading R16) on BASELINE config 1 against the oracle's own
    two-stage retrieval on dense LU solves (run here, and as stored by tests/golden/make_oracle_goldens.py)."""
    geo = wl.sphere_lattice((7, 7, 7))
    c = coeffs(geo)

    def xi_oracle(kappa):
        return np.array([orc.zero_order(orc.solve_dense(c, geo.periods, geo.orders, np.array([0, 0, kv]), TWO_PI,
                                                        geo.eps_b, [1.0, 0, 0]))[0] for kv in kappa])
    n_o, eps_o, zeta_o = orc.retrieve_two_stage(xi_oracle, TWO_PI, 1.02, 1.30)
    plan = gsm.plan_from_geometry(geo, max_iters=100, max_batch=32)
    n_g, eps_g, zeta_g, st = plan.retrieve_neff([0, 0, 1.0], [1.0, 0, 0], 0, TWO_PI, 1.02, 1.30, tol=1e-12)
    assert st == gsm.OK
    assert abs(eps_g - eps_o) <= 1e-8 and abs(n_g - n_o) <= 1e-8
    assert abs(zeta_g - zeta_o) <= 1e-6 * abs(zeta_o)
    gold = load_oracle_golden()
    assert abs(n_g.real - gold["cfg1_7_zx_neff_re"]) <= 1e-8 and abs(n_g.imag) <= 1e-9
    assert abs(eps_g.real - gold["cfg1_7_zx_eps_re"]) <= 1e-8
    with pytest.raises(gsm.GsmError):          # an odd fine mesh would put a node on the estimate: rejected
        plan.retrieve_neff([0, 0, 1.0], [1.0, 0, 0], 0, TWO_PI, 1.02, 1.30, nfine=17, tol=1e-10)
    plan.close()


def test_retrieve_neff_config3_tensor_entries():
    """BASELINE config 3: the three diagonal entries of eps_eff (reading R14) at 15^3 orders through gsm_retrieve_neff
    against the oracle's own two-stage retrieval (tests/golden/oracle_neff.txt, written by make_oracle_goldens.py)."""
    geo = wl.ellipsoid_lattice((15, 15, 15))
    plan = gsm.plan_from_geometry(geo, max_iters=120, max_batch=32)
    gold = load_oracle_golden()
    for key, (pa, qa) in wl.DIRECTIONS.items():
        d = np.zeros(3); d[pa] = 1.0
        pol = np.zeros(3, dtype=complex); pol[qa] = 1.0
        n, eps, zeta, st = plan.retrieve_neff(d, pol, qa, TWO_PI, 1.02, 1.30, tol=1e-12)
        assert st == gsm.OK and abs(n.imag) <= 1e-9
        assert abs(n.real - gold[f"cfg3_15_{key}_neff_re"]) <= 1e-8 and abs(eps.real - gold[f"cfg3_15_{key}_eps_re"]) <= 1e-8
        assert abs(eps - n * n) <= 1e-14
    plan.close()
