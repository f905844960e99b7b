"""Pins for the CPU oracle (oracle/gsm_oracle.py): each test checks it against something OTHER than itself -
closed forms, quadrature, literal brute-force loops, invariants, textbook eigenproblems (CPU only)."""
import itertools
import math

import numpy as np
import pytest
import scipy.integrate
import scipy.linalg
import scipy.optimize

from oracle import gsm_oracle as O
from paper_1501_01752_b200 import workloads as W

K0 = 2 * np.pi


def coeffs(g):
    return O.coeffs_analytic(g.periods, g.orders, g.shapes, g.eps_bg, g.eps_b)


# ---- a0: harmonics ----------------------------------------------------------------------------------
def test_sphere_coefficients_vs_radial_quadrature():
    """c_d of a centred sphere = Delta (4 pi / V) int_0^R r^2 sinc(|G_d| r) dr (independent of the closed form)."""
    g = W.sphere_lattice((5, 5, 5))
    c = coeffs(g)
    L, R, delta = g.periods[0], g.shapes[0]["size"][0], (4.0 - 1.0) / 1.0
    for d in [(0, 0, 0), (1, 0, 0), (1, 2, 0), (2, 2, 1), (4, 4, 4), (-3, 2, -4)]:
        G = 2 * np.pi / L * math.sqrt(sum(t * t for t in d))
        val, _ = scipy.integrate.quad(lambda r: r * r * (np.sinc(G * r / np.pi)), 0, R, epsabs=1e-15, epsrel=1e-13)
        ref = delta * 4 * np.pi * val / L**3
        got = c[d[0] + 4, d[1] + 4, d[2] + 4]
        assert abs(got - ref) < 1e-13
    f = 4 / 3 * np.pi * R**3 / L**3
    assert abs(c[4, 4, 4] - f * delta) < 1e-15                          # c_0 = f Delta
    assert np.allclose(c, np.conj(c[::-1, ::-1, ::-1]), atol=1e-16)     # c_{-d} = conj c_d
    assert np.abs(c.imag).max() < 1e-16                                 # centred => real


def test_sphere_closed_form_vs_direct_dft_of_voxelised_sphere():
    """Direct DFT of a voxelised sphere converges to the closed form as the grid refines."""
    orders = (3, 3, 3)
    g = W.sphere_lattice(orders)
    c = coeffs(g)
    L, R = g.periods[0], g.shapes[0]["size"][0]
    errs = []
    for nv in (12, 48, 128):
        ax = np.arange(nv) * L / nv
        d = np.minimum(ax, L - ax)
        r2 = d[:, None, None] ** 2 + d[None, :, None] ** 2 + d[None, None, :] ** 2
        grid = np.where(r2 <= R * R, 4.0, 1.0)
        cv = O.coeffs_voxel(grid, orders, 1.0)
        errs.append(np.abs(cv - c).max())
    assert errs[0] > errs[1] > errs[2] and errs[2] < 2e-4


def test_shifted_and_box_coefficients():
    """Laminate f sinc(pi d f) vanishes at even d for f = 0.5; a half-period shift multiplies c_d by (-1)^d."""
    g = W.laminate((1, 1, 15))
    c = coeffs(g)[0, 0]
    d = np.arange(-14, 15)
    ref = 8.0 * 0.5 * np.sinc(d * 0.5)
    assert np.allclose(c, ref, atol=1e-15)
    assert np.abs(c[(d % 2 == 0) & (d != 0)]).max() < 1e-15
    sh = [dict(kind=W.BOX, center=(0, 0, 0.5), size=(1, 1, 0.5), eps=9.0)]
    c2 = O.coeffs_analytic(g.periods, g.orders, sh, 1.0, 1.0)[0, 0]
    assert np.allclose(c2, c * (-1.0) ** np.abs(d), atol=1e-14)
    # box coefficient along one axis vs quadrature of exp(-iGz) over the slab
    w = 0.3
    sh = [dict(kind=W.BOX, center=(0, 0, 0.1), size=(1, 1, w), eps=3.0)]
    c3 = O.coeffs_analytic((1, 1, 1), (1, 1, 4), sh, 1.0, 1.0)[0, 0]
    for dd in range(-3, 4):
        re, _ = scipy.integrate.quad(lambda z: np.cos(2 * np.pi * dd * z), 0.1 - w / 2, 0.1 + w / 2)
        im, _ = scipy.integrate.quad(lambda z: -np.sin(2 * np.pi * dd * z), 0.1 - w / 2, 0.1 + w / 2)
        assert abs(c3[dd + 3] - 2.0 * (re + 1j * im)) < 1e-13


def test_eps_b_offset_term():
    """eps_b != eps_bg adds (eps_bg-eps_b)/eps_b at d=0 and rescales the contrast by 1/eps_b."""
    g = W.sphere_lattice((3, 3, 3))
    c1 = O.coeffs_analytic(g.periods, g.orders, g.shapes, 1.0, 1.0)
    c2 = O.coeffs_analytic(g.periods, g.orders, g.shapes, 1.0, 1.6)
    ref = c1 / 1.6
    ref[2, 2, 2] += (1.0 - 1.6) / 1.6
    assert np.allclose(c2, ref, atol=1e-15)


def test_ellipsoid_coefficients_pinned():
    """ELLIPSOID branch of coeffs_analytic (config 3 rests on it), pinned four ways:
    (1) radial quadrature: the affine map r = s o u turns the ellipsoid into the unit ball, so
        c_d = Delta (4 pi a b c / V) int_0^1 u^2 sinc(|G o s| u) du exp(-i G.r_c) - independent of the closed form;
    (2) direct DFT of a voxelised off-centre ellipsoid converges to it as the grid refines;
    (3) a = b = c reduces to the sphere coefficients; (4) c_0 = f Delta with f = 4 pi a b c / (3 V)."""
    per, orders = (0.2, 0.25, 0.3), (3, 3, 3)
    semi, ctr, eps_i = (0.07, 0.05, 0.04), (0.03, -0.02, 0.05), 12.0
    sh = [dict(kind=W.ELLIPSOID, center=ctr, size=semi, eps=eps_i)]
    c = O.coeffs_analytic(per, orders, sh, 1.0, 1.0)
    V = per[0] * per[1] * per[2]
    delta = eps_i - 1.0
    for d in itertools.product(range(-2, 3), repeat=3):
        G = [2 * np.pi * d[a] / per[a] for a in range(3)]
        x = math.sqrt(sum((G[a] * semi[a]) ** 2 for a in range(3)))
        val, _ = scipy.integrate.quad(lambda u: u * u * np.sinc(x * u / np.pi), 0, 1, epsabs=1e-15, epsrel=1e-13)
        ref = delta * 4 * np.pi * semi[0] * semi[1] * semi[2] * val / V * np.exp(-1j * sum(G[a] * ctr[a] for a in range(3)))
        assert abs(c[d[0] + 2, d[1] + 2, d[2] + 2] - ref) < 1e-13
    assert abs(c[2, 2, 2] - delta * 4 / 3 * np.pi * semi[0] * semi[1] * semi[2] / V) < 1e-15
    assert np.allclose(c, np.conj(c[::-1, ::-1, ::-1]), atol=1e-16)
    errs = []
    for nv in (16, 48, 96):
        ax = [np.arange(nv) * per[a] / nv for a in range(3)]
        dd = []
        for a in range(3):
            t = (ax[a] - ctr[a] + per[a] / 2) % per[a] - per[a] / 2          # minimum-image offset from the centre
            dd.append((t / semi[a]) ** 2)
        inside = dd[0][:, None, None] + dd[1][None, :, None] + dd[2][None, None, :] <= 1.0
        cv = O.coeffs_voxel(np.where(inside, eps_i, 1.0), orders, 1.0)
        errs.append(np.abs(cv - c).max())
    assert errs[0] > errs[1] > errs[2] and errs[2] < 5e-3 * abs(c[2, 2, 2])
    R = 0.06
    cs = O.coeffs_analytic(per, orders, [dict(kind=W.SPHERE, center=ctr, size=(R, 0, 0), eps=eps_i)], 1.0, 1.0)
    ce = O.coeffs_analytic(per, orders, [dict(kind=W.ELLIPSOID, center=ctr, size=(R, R, R), eps=eps_i)], 1.0, 1.0)
    assert np.max(np.abs(cs - ce)) < 1e-15                     # same numbers up to the rounding of |G| R vs |G o s|


def test_voxel_dft_separable_vs_literal_triple_sum():
    rng = np.random.default_rng(3)
    grid = rng.uniform(1, 5, (4, 5, 6)) + 1j * rng.uniform(0, 1, (4, 5, 6))
    orders = (2, 3, 3)
    cv = O.coeffs_voxel(grid, orders, 1.3)
    for d in itertools.product(range(-1, 2), range(-2, 3), range(-2, 3)):
        assert abs(cv[d[0] + 1, d[1] + 2, d[2] + 2] - O.coeffs_voxel_single(grid, d, 1.3)) < 1e-14


# ---- a1-a4: Toeplitz product --------------------------------------------------------------------------
def _literal_toeplitz(c, x):
    """Brute force with explicit harmonic indices m, m' (independent index arithmetic)."""
    N = x.shape[1:]
    rng = [O.order_range(n) for n in N]
    y = np.zeros_like(x)
    for a, m1 in enumerate(rng[0]):
        for b, m2 in enumerate(rng[1]):
            for cc, m3 in enumerate(rng[2]):
                for a2, p1 in enumerate(rng[0]):
                    for b2, p2 in enumerate(rng[1]):
                        for c2, p3 in enumerate(rng[2]):
                            coef = c[(m1 - p1) + N[0] - 1, (m2 - p2) + N[1] - 1, (m3 - p3) + N[2] - 1]
                            y[:, a, b, cc] += coef * x[:, a2, b2, c2]
    return y


@pytest.mark.parametrize("orders", [(3, 3, 3), (2, 3, 4), (1, 1, 7)])
def test_toeplitz_matvec_vs_literal_loops(orders):
    rng = np.random.default_rng(1)
    c = rng.standard_normal([2 * n - 1 for n in orders]) + 1j * rng.standard_normal([2 * n - 1 for n in orders])
    x = W.random_field(1, orders)[0]
    ref = _literal_toeplitz(c, x)
    assert np.allclose(O.toeplitz_matvec(c, x), ref, atol=1e-13)
    assert np.allclose(O.toeplitz_matvec_c(c, x), ref, atol=1e-13)


def test_toeplitz_unit_vector_returns_column_of_c():
    orders = (3, 5, 4)
    rng = np.random.default_rng(2)
    c = rng.standard_normal([2 * n - 1 for n in orders]) + 0j
    x = np.zeros((3,) + orders, complex)
    j = (1, 3, 2)
    x[(1,) + j] = 1.0
    y = O.toeplitz_matvec(c, x)
    for i in itertools.product(*[range(n) for n in orders]):
        d = [i[a] - j[a] + orders[a] - 1 for a in range(3)]
        assert y[(1,) + i] == c[tuple(d)]
    assert np.all(y[0] == 0) and np.all(y[2] == 0)


def test_c_matvec_matches_numpy_at_15cubed():
    g = W.ellipsoid_lattice((15, 15, 15))
    c = coeffs(g)
    x = W.random_field(1, g.orders)[0]
    y = O.toeplitz_matvec_c(c, x)
    for i in [(0, 0, 0), (14, 14, 14), (7, 3, 11), (2, 13, 5)]:
        assert np.allclose(y[(slice(None),) + i], O.toeplitz_row(c, x, i), rtol=0, atol=1e-12)


# ---- a5: Green dyadic ---------------------------------------------------------------------------------
def test_green_dyadic_eigen_identities():
    """G_m k_m = -k_m; G_m t = k_b^2/(k_m^2-k_b^2) t for t perpendicular to k_m; G symmetric."""
    periods, orders = (0.2, 0.25, 0.3), (3, 3, 3)
    k_inc, k0, eps_b = np.array([0.3, -0.2, 1.1]) * K0, K0, 1.7
    k = O.wavevectors(periods, orders, k_inc)
    kb2 = k0 * k0 * eps_b
    assert np.allclose(O.green_multiply(k.astype(complex), periods, k_inc, k0, eps_b), -k, atol=1e-12)
    t = np.cross(k, np.array([0.3, 0.5, -0.2])[:, None, None, None], axis=0).astype(complex)
    lam = kb2 / ((k**2).sum(0) - kb2)
    assert np.allclose(O.green_multiply(t, periods, k_inc, k0, eps_b), lam[None] * t, atol=1e-12)
    rng = np.random.default_rng(0)
    u, v = rng.standard_normal((2, 3) + orders)
    Gu = O.green_multiply(u.astype(complex), periods, k_inc, k0, eps_b)
    Gv = O.green_multiply(v.astype(complex), periods, k_inc, k0, eps_b)
    assert np.allclose((v * Gu).sum(0), (u * Gv).sum(0), atol=1e-12)     # v.G u = u.G v per harmonic


# ---- solves ------------------------------------------------------------------------------------------
def test_homogeneous_cell_is_identity_and_lucky_breakdown():
    """Delta eps = 0 => A = I, E = E_inc exactly, GMRES stops after one iteration without dividing by zero."""
    g = W.sphere_lattice((3, 3, 3), eps=1.0)
    c = coeffs(g)
    assert np.all(c == 0)
    E, hist, m = O.solve_gmres(c, g.periods, g.orders, np.array([0, 0, 1.2 * K0]), K0, 1.0, [1, 0, 0], tol=1e-12)
    assert m == 1 and hist[0] == 0.0
    assert np.array_equal(E, O.incident(g.orders, [1, 0, 0]))
    assert np.all(np.isfinite(E))


def test_uniform_cell_closed_form():
    """c_d = Delta delta_d0: transverse E_0 = a (kappa^2-k0^2 eps_b)/(kappa^2-k0^2 eps_2); longitudinal a eps_b/eps_2."""
    orders, periods, eps_b, eps_2 = (3, 3, 3), (0.2, 0.2, 0.2), 1.0, 2.5
    box = [dict(kind=W.BOX, center=(0, 0, 0), size=periods, eps=eps_2)]
    c = O.coeffs_analytic(periods, orders, box, 1.0, eps_b)
    assert abs(c[2, 2, 2] - 1.5) < 1e-15 and np.abs(np.delete(c.ravel(), 62)).max() < 1e-15
    kap = 1.3 * K0
    E = O.solve_dense(c, periods, orders, np.array([0, 0, kap]), K0, eps_b, [1, 0, 0])
    ref = (kap**2 - K0**2 * eps_b) / (kap**2 - K0**2 * eps_2)
    assert abs(O.zero_order(E)[0] - ref) < 1e-13
    assert np.abs(E).sum() - abs(O.zero_order(E)[0]) < 1e-12          # only m = 0 is excited
    E = O.solve_dense(c, periods, orders, np.array([0, 0, kap]), K0, eps_b, [0, 0, 1])
    assert abs(O.zero_order(E)[2] - eps_b / eps_2) < 1e-13


@pytest.mark.parametrize("orders", [(3, 3, 3), (5, 5, 5), (1, 1, 31)])
def test_gmres_matches_dense_lu(orders):
    g = W.sphere_lattice(orders) if orders[0] > 1 else W.laminate(orders)
    c = coeffs(g)
    k_inc = np.array([0.0, 0.0, 1.2 * K0]) if orders[0] > 1 else np.array([0.0, 0.0, 0.9])
    k0 = K0 if orders[0] > 1 else 0.5
    E1 = O.solve_dense(c, g.periods, g.orders, k_inc, k0, g.eps_b, [1, 0, 0])
    E2, hist, m = O.solve_gmres(c, g.periods, g.orders, k_inc, k0, g.eps_b, [1, 0, 0], tol=1e-13)
    assert np.linalg.norm(E1 - E2) / np.linalg.norm(E1) < 1e-11
    assert all(hist[i + 1] <= hist[i] * (1 + 1e-12) for i in range(len(hist) - 1))     # non-increasing
    r = O.incident(g.orders, [1, 0, 0]) - O.apply_operator(c, E2, g.periods, k_inc, k0, g.eps_b)
    assert abs(np.linalg.norm(r) - hist[-1]) < 1e-12                                   # estimate = true residual
    if orders[0] > 1:
        assert np.abs(E2.imag).max() < 1e-13                                           # real c, real kappa => real E


def test_dense_assembly_matches_operator():
    g = W.ellipsoid_lattice((3, 3, 3))
    c = coeffs(g)
    k_inc = np.array([0.1, 0.2, 1.1]) * K0
    A = O.assemble_dense(c, g.periods, g.orders, k_inc, K0, 1.0 + 0.2j)
    x = W.random_field(1, g.orders)[0]
    y = O.apply_operator(c, x, g.periods, k_inc, K0, 1.0 + 0.2j)
    assert np.allclose(A @ x.ravel(), y.ravel(), atol=1e-12)


# ---- poles -------------------------------------------------------------------------------------------
def test_pole_search_recovers_synthetic_poles():
    eta = np.array([1.37 + 0.002j, 0.4 - 0.1j])
    zeta = np.array([0.6 - 0.1j, 0.05 + 0.02j])
    kap = np.linspace(1.2, 1.5, 16)
    xi = sum(z / (kap - e) for z, e in zip(zeta, eta)) + 0.3 - 0.2 * kap + 0.05j * kap**2
    e, z = O.pole_search(kap, xi, 5, 10)
    j = O.select_pole(e, z, 1.2, 1.5)
    assert abs(e[j] - eta[0]) < 1e-10 and abs(z[j] - zeta[0]) < 1e-9


def _scan_pole(g, c, kap, prop, pol, k0, eps_b, solver):
    xi = []
    for kp in kap:
        k_inc = np.zeros(3)
        k_inc[prop] = kp
        a = np.zeros(3)
        a[pol] = 1.0
        xi.append(O.zero_order(solver(c, g.periods, g.orders, k_inc, k0, eps_b, a))[pol])
    eta, zeta = O.pole_search(kap, xi, 5, 10)
    j = O.select_pole(eta, zeta, kap[0], kap[-1])
    assert j >= 0
    return eta[j], zeta[j]


def test_pole_is_eigenvalue_of_hermitian_pencil_and_independent_of_eps_b():
    """At k_inc = eta z, k0^2 is a generalised eigenvalue of (k_m^2 I - k_m k_m^T) E = k0^2 [eps] E (textbook
    plane-wave eigenproblem); and the pole does not move when eps_b changes (exact in the truncated system)."""
    g = W.sphere_lattice((5, 5, 5))
    kap = W.kappa_mesh(1.04, 1.16, 15) + 0.0007
    poles = []
    for eps_b in (1.0, 1.6):
        c = O.coeffs_analytic(g.periods, g.orders, g.shapes, 1.0, eps_b)
        eta, _ = _scan_pole(g, c, kap, 2, 0, K0, eps_b, O.solve_dense)
        poles.append(eta)
    assert abs(poles[0] - poles[1]) < 1e-8 * K0
    eta = poles[0].real
    c = O.coeffs_analytic(g.periods, g.orders, g.shapes, 1.0, 1.0)
    N, n = g.orders, g.n
    idx = np.array(list(itertools.product(*[range(t) for t in N])))
    Teps = c[idx[:, None, 0] - idx[None, :, 0] + N[0] - 1, idx[:, None, 1] - idx[None, :, 1] + N[1] - 1,
             idx[:, None, 2] - idx[None, :, 2] + N[2] - 1] + np.eye(n)
    k = O.wavevectors(g.periods, N, np.array([0, 0, eta])).reshape(3, n)
    M = np.zeros((3 * n, 3 * n), complex)
    B = np.zeros((3 * n, 3 * n), complex)
    for a in range(3):
        B[a * n:(a + 1) * n, a * n:(a + 1) * n] = Teps
        for b in range(3):
            M[a * n:(a + 1) * n, b * n:(b + 1) * n] = np.diag(((k**2).sum(0) if a == b else 0.0) - k[a] * k[b])
    w = scipy.linalg.eigh(M, B, eigvals_only=True)
    w = w[w > 1e-6]
    assert abs(np.sqrt(w.min()) / K0 - 1.0) < 1e-8


# ---- laminate vs Rytov -------------------------------------------------------------------------------
def rytov_bloch_K(k0, e1, e2, d1, d2):
    """cos K L = cos k1d1 cos k2d2 - 1/2 (k1/k2 + k2/k1) sin k1d1 sin k2d2, normal incidence (textbook, Rytov 1956)."""
    k1, k2 = k0 * math.sqrt(e1), k0 * math.sqrt(e2)
    rhs = math.cos(k1 * d1) * math.cos(k2 * d2) - 0.5 * (k1 / k2 + k2 / k1) * math.sin(k1 * d1) * math.sin(k2 * d2)
    return math.acos(rhs) / (d1 + d2)


def rytov_inplane_beta(k0, e1, e2, d1, d2, tm):
    """In-plane propagation (K_z = 0): 1 = cos q1d1 cos q2d2 - 1/2 (p + 1/p) sin q1d1 sin q2d2,
    q_i = sqrt(k0^2 e_i - beta^2), p = q1/q2 (TE) or e2 q1/(e1 q2) (TM); fundamental root."""
    def f(beta):
        q1, q2 = np.sqrt(complex(k0 * k0 * e1 - beta * beta)), np.sqrt(complex(k0 * k0 * e2 - beta * beta))
        p = q1 / q2 * ((e2 / e1) if tm else 1.0)
        return (np.cos(q1 * d1) * np.cos(q2 * d2) - 0.5 * (p + 1 / p) * np.sin(q1 * d1) * np.sin(q2 * d2) - 1.0).real
    lo, hi = k0 * math.sqrt(min(e1, e2)) * 1.0001, k0 * math.sqrt(max(e1, e2)) * 0.9999
    return scipy.optimize.brentq(f, lo, hi, xtol=1e-15, rtol=1e-15)


@pytest.mark.parametrize("lam_ratio", [0.01, 0.1, 0.17])
def test_laminate_normal_incidence_matches_rytov(lam_ratio):
    g = W.laminate((1, 1, 63))
    c = coeffs(g)
    k0 = 2 * np.pi * lam_ratio                     # length unit = Lambda_z
    K = rytov_bloch_K(k0, 1.0, 9.0, 0.5, 0.5)
    h = 0.004 * K
    kap = K + h * (np.arange(15) - 7 + 0.5)        # pole mid-way between two nodes (R16)
    eta, _ = _scan_pole(g, c, kap, 2, 0, k0, 1.0, O.solve_dense)
    assert abs(eta.imag) < 1e-9 * K
    assert abs(eta.real / K - 1.0) < 2e-6          # truncation error ~ N^-3


def test_laminate_long_wavelength_limits():
    """Lambda/lambda = 0.01: eps_TE -> arithmetic mean 5 (Rytov 5.0013); TM (Laurent rule) converges to the
    harmonic-mean side only as 1/N - check the 1/N trend toward Rytov's TM value."""
    k0 = 2 * np.pi * 0.01
    bte = rytov_inplane_beta(k0, 1.0, 9.0, 0.5, 0.5, tm=False)
    btm = rytov_inplane_beta(k0, 1.0, 9.0, 0.5, 0.5, tm=True)
    assert abs((bte / k0) ** 2 - 5.0) < 2e-3 and abs((btm / k0) ** 2 - 1.8) < 1e-3
    g = W.laminate((1, 1, 63))
    c = coeffs(g)
    kap = bte * (1 + 0.004 * (np.arange(15) - 7 + 0.5))
    eta, _ = _scan_pole(g, c, kap, 0, 1, k0, 1.0, O.solve_dense)          # k || x, a = y  (TE)
    assert abs((eta.real / k0) ** 2 - (bte / k0) ** 2) < 1e-7
    errs = []
    for N3 in (15, 31, 63):
        g = W.laminate((1, 1, N3))
        c = coeffs(g)
        kap = np.linspace(1.30, 1.60, 16) * k0
        eta, _ = _scan_pole(g, c, kap, 0, 2, k0, 1.0, O.solve_dense)      # k || x, a = z  (TM)
        errs.append(abs(eta.real - btm) / k0)
    assert errs[0] > errs[1] > errs[2]
    assert 1.6 < errs[0] / errs[1] < 2.6 and 1.6 < errs[1] / errs[2] < 2.6   # ~1/N


def test_two_stage_retrieval_synthetic_pole_and_uniform_cell():
    """retrieve_two_stage (reading R16) recovers a known pole of a synthetic meromorphic response, and for the uniform
    cell (closed form: pole at kappa = k0 sqrt(eps_2)) returns n_eff = sqrt(eps_2), eps_eff = eps_2."""
    import numpy as np
    from oracle import gsm_oracle as orc
    k0 = 2.0 * np.pi
    eta_true, zeta_true = 1.2345678 * k0 + 0.0j, 0.37 - 0.11j

    def xi(kappa):
        return zeta_true / (kappa - eta_true) + 0.3 - 0.02 * kappa + 0.004 * kappa**2 + 0.05 / (kappa + 9.0)
    n, eps, zeta = orc.retrieve_two_stage(xi, k0, 1.05, 1.45)
    assert abs(n - 1.2345678) <= 1e-11 and abs(eps - 1.2345678**2) <= 1e-10 and abs(zeta - zeta_true) <= 1e-8

    eps2 = 2.5
    shapes = [dict(kind=orc.BOX, center=(0, 0, 0), size=(0.2, 0.2, 0.2), eps=eps2)]
    c = orc.coeffs_analytic((0.2, 0.2, 0.2), (3, 3, 3), shapes, 1.0, 1.0)

    def xi_cell(kappa):
        return np.array([orc.zero_order(orc.solve_dense(c, (0.2, 0.2, 0.2), (3, 3, 3), np.array([0, 0, kv]), k0, 1.0,
                                                        [1.0, 0, 0]))[0] for kv in kappa])
    n, eps, _ = orc.retrieve_two_stage(xi_cell, k0, 1.3, 1.8)
    assert abs(eps - eps2) <= 1e-9 and abs(n - np.sqrt(eps2)) <= 1e-9


def test_gmres_with_initial_guess():
    """gmres(x0=...) (Saad Alg. 6.9 with a non-zero start): same solution as dense LU whatever the guess;
    the exact solution as guess takes no iteration; the neighbouring kappa point's field as guess takes fewer iterations
    than the zero start; the history stays relative to ||b||."""
    g = W.sphere_lattice((5, 5, 5))
    c = coeffs(g)
    kb, kb2 = np.array([0.0, 0.0, 1.12 * K0]), np.array([0.0, 0.0, 1.125 * K0])
    pol = [1.0, 0.2j, 0.0]
    ref = O.solve_dense(c, g.periods, g.orders, kb, K0, 1.0, pol)
    nb = O.solve_dense(c, g.periods, g.orders, kb2, K0, 1.0, pol)
    E0, h0, m0 = O.solve_gmres(c, g.periods, g.orders, kb, K0, 1.0, pol, tol=1e-12)
    rnd = W.random_field(1, g.orders)[0]
    for x0 in (nb, rnd, 3.0 * ref):
        E, h, m = O.solve_gmres(c, g.periods, g.orders, kb, K0, 1.0, pol, tol=1e-12, x0=x0)
        assert np.linalg.norm(E - ref) / np.linalg.norm(ref) < 1e-10
        assert h[-1] <= 1e-12 and np.all(np.diff(h) <= 1e-15)
        r = O.incident(g.orders, pol) - O.apply_operator(c, E, g.periods, kb, K0, 1.0)
        assert abs(np.linalg.norm(r) / np.linalg.norm(O.incident(g.orders, pol)) - h[-1]) < 1e-12   # estimate = true, / ||b||
    E, h, m = O.solve_gmres(c, g.periods, g.orders, kb, K0, 1.0, pol, tol=1e-12, x0=nb)
    assert m < m0
    E, h, m = O.solve_gmres(c, g.periods, g.orders, kb, K0, 1.0, pol, tol=1e-10, x0=ref)
    assert m == 0 and h == [] and np.array_equal(E, ref)


# ---- a0: polyhedron Fourier image -----------------------------------------------------
def test_polyhedron_image_pinned():
    """polyhedron_image against things other than itself: (1) an axis-aligned cube is the box closed form (product of
    sincs) - exercises the G_t = 0 branch; (2) volumes at G = 0 (tetrahedron 8/3 s^3, octahedron 4/3 s^3, L-prism 3 s^3);
    (3) a rotated tetrahedron against adaptive cubature over its volume (scipy tplquad on the affine image of the unit
    simplex); (4) a translation multiplies by exp(-i G.t); (5) reversing the face orientation flips the sign;
    (6) the L-shaped (non-convex) prism equals the difference of two boxes."""
    v, f = W.polyhedron("cube", 0.03)
    for G in [(0, 0, 0), (31.4, 0, 0), (31.4, -62.8, 0), (10.0, 20.0, -35.0), (0, 0, 94.2)]:
        ref = 0.06**3 * np.prod([np.sinc(g * 0.03 / np.pi) for g in G])
        assert abs(O.polyhedron_image(G, v, f) - ref) < 1e-15 * 0.06**3 * 100
    s = 0.07
    assert abs(O.polyhedron_image((0, 0, 0), *W.polyhedron("tetrahedron", s)) - 8 / 3 * s**3) < 1e-18
    assert abs(O.polyhedron_image((0, 0, 0), *W.polyhedron("octahedron", s)) - 4 / 3 * s**3) < 1e-18
    assert abs(O.polyhedron_image((0, 0, 0), *W.polyhedron("lshape", s)) - 3 * s**3) < 1e-18
    v, f = W.polyhedron("tetrahedron", s, rotate=((1.0, 2.0, 3.0), 0.4))
    M = np.stack([v[1] - v[0], v[2] - v[0], v[3] - v[0]], axis=1)          # r = v0 + M (a, b, c) on the unit simplex
    jac = abs(np.linalg.det(M))
    for G in [np.array([31.4, 0.0, 0.0]), np.array([-20.0, 45.0, 12.0])]:
        def integrand(c, b, a, part):
            ph = -G @ (v[0] + M @ np.array([a, b, c]))
            return math.cos(ph) if part == 0 else math.sin(ph)
        val = [scipy.integrate.tplquad(integrand, 0, 1, lambda a: 0, lambda a: 1 - a, lambda a, b: 0, lambda a, b: 1 - a - b,
                                       args=(part,), epsabs=1e-13, epsrel=1e-11)[0] for part in (0, 1)]
        assert abs(O.polyhedron_image(G, v, f) - jac * (val[0] + 1j * val[1])) < 1e-11 * jac
        t = np.array([0.01, -0.02, 0.015])
        assert abs(O.polyhedron_image(G, v + t, f) - np.exp(-1j * G @ t) * O.polyhedron_image(G, v, f)) < 1e-18
        assert abs(O.polyhedron_image(G, v, [tuple(reversed(q)) for q in f]) + O.polyhedron_image(G, v, f)) < 1e-17
    v, f = W.polyhedron("lshape", s)
    for G in [(31.4, 0, 0), (10.0, -20.0, 30.0), (0.0, 62.8, 31.4)]:
        G = np.array(G)
        big = (2 * s) ** 2 * s * np.prod([np.sinc(g * w / 2 / np.pi) for g, w in zip(G, (2 * s, 2 * s, s))])
        cut = s * s * s * np.prod([np.sinc(g * s / 2 / np.pi) for g in G]) * np.exp(-1j * (G[0] + G[1]) * s / 2)
        assert abs(O.polyhedron_image(G, v, f) - (big - cut)) < 1e-16 * 100


def test_polyhedron_coefficients_vs_voxelised_direct_dft():
    """coeffs_analytic with a rotated off-centre octahedron: direct DFT of its voxelisation converges to it; c_0 = f Delta;
    Hermitian symmetry."""
    g = W.polyhedron_lattice((3, 3, 3), "octahedron", center=(0.02, -0.01, 0.03))
    c = coeffs(g)
    sh = g.shapes[0]
    L = g.periods[0]
    assert abs(c[2, 2, 2] - (sh["eps"] - 1.0) * 4 / 3 * 0.07**3 / L**3) < 1e-15
    assert np.allclose(c, np.conj(c[::-1, ::-1, ::-1]), atol=1e-16)
    v, faces = sh["vertices"], sh["faces"]
    normals, offs = [], []
    for f in faces:                                   # inside <=> n_f.(r - v_f) <= 0 for every face (convex)
        n = np.cross(v[f[1]] - v[f[0]], v[f[2]] - v[f[0]])
        normals.append(n / np.linalg.norm(n)); offs.append(normals[-1] @ v[f[0]])
    errs = []
    for nv in (16, 48, 96):
        ax = np.arange(nv) * L / nv
        r = np.stack(np.meshgrid(ax, ax, ax, indexing="ij"), axis=-1) - np.asarray(sh["center"])
        r = (r + L / 2) % L - L / 2                   # minimum image
        inside = np.ones((nv, nv, nv), dtype=bool)
        for n, o in zip(normals, offs):
            inside &= (r @ n) <= o
        errs.append(np.abs(O.coeffs_voxel(np.where(inside, sh["eps"], 1.0), g.orders, 1.0) - c).max())
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1e-2 * abs(c[2, 2, 2])


def test_gmres_guess_off_by_one_eigenvector_breaks_down_after_one_iteration():
    """Reading R23 with a guessed start.  Uniform cell: A is block diagonal over the harmonics and a unit vector u at
    harmonic m = (1, 0, 0) polarised along y (transverse to k_m) is an eigenvector.  x0 = x* + 1e-7 u gives r0 parallel
    to u, so the Krylov space is one-dimensional: A v_0 has nothing left after orthogonalisation and GMRES must stop
    after ONE iteration at the exact solution, even with a tolerance that can never be met.  ||r0|| is 1e-7 ||b|| here:
    a breakdown test scaled by ||r0|| would miss it and go on dividing by a rounding-level h_{j+1,j}."""
    eps2 = 2.5
    g = W.Geometry("uniform", (0.2, 0.2, 0.2), (3, 3, 3),
                   [dict(kind=W.BOX, center=(0, 0, 0), size=(0.2, 0.2, 0.2), eps=eps2)], 1.0, 1.0, None, ())
    c = coeffs(g)
    kb, pol = np.array([0.0, 0.0, 1.3 * K0]), [1.0, 0.0, 0.0]
    ref = O.solve_dense(c, g.periods, g.orders, kb, K0, 1.0, pol)
    u = np.zeros_like(ref)
    u[1, 2, 1, 1] = 1.0                                   # component y at m = (+1, 0, 0)
    lam = (O.apply_operator(c, u, g.periods, kb, K0, 1.0))[1, 2, 1, 1]
    assert np.linalg.norm(O.apply_operator(c, u, g.periods, kb, K0, 1.0) - lam * u) < 1e-14      # u is an eigenvector
    E, h, m = O.solve_gmres(c, g.periods, g.orders, kb, K0, 1.0, pol, tol=1e-30, max_iters=20, x0=ref + 1e-7 * u)
    assert m == 1 and np.linalg.norm(E - ref) / np.linalg.norm(ref) < 1e-14
