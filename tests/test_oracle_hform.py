"""Pins of the oracle's H-field formulation (Eq. 5) against things other than itself:
closed forms, an invariant, two independent statements of the operator (Levi-Civita sums vs cross products), the
textbook Hermitian plane-wave eigenproblem at the pole, dense LU vs GMRES, and the Rytov laminate dispersion."""
import numpy as np

from oracle import gsm_oracle as orc
from paper_1501_01752_b200 import workloads as wl

TWO_PI = 2.0 * np.pi


def D_of(geo):
    return orc.coeffs_inverse_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)


def test_inverse_permittivity_coefficients_closed_form_vs_voxel_dft():
    geo = wl.sphere_lattice((3, 3, 3))
    D = D_of(geo)
    f = 4.0 / 3.0 * np.pi * 0.3**3
    assert abs(D[2, 2, 2] - (1.0 - 1.0 / 4.0) * f) <= 1e-15           # D_0 = f (eps_b/eps_bg - eps_b/eps_i)
    assert np.allclose(D, np.conj(D[::-1, ::-1, ::-1]), atol=1e-15)    # real 1/eps -> Hermitian coefficients
    errs = []
    for nv in (24, 48):
        ax = np.arange(nv) * (0.2 / nv)
        d = np.minimum(ax, 0.2 - ax)
        r2 = d[:, None, None] ** 2 + d[None, :, None] ** 2 + d[None, None, :] ** 2
        grid = np.where(r2 <= 0.06**2, 4.0, 1.0).astype(complex)
        errs.append(np.abs(orc.coeffs_inverse_voxel(grid, geo.orders, 1.0) - D).max())
    assert errs[1] < errs[0] and errs[1] <= 5e-4
    # complex eps_b, lossy inclusion, off-centre box: D = 1 - eps_b/eps sampled exactly when the box fits the voxels
    box = [dict(kind=wl.BOX, center=(0.05, 0.0, 0.0), size=(0.1, 0.2, 0.1), eps=3.0 + 0.2j)]
    Db = orc.coeffs_inverse_analytic((0.2, 0.2, 0.2), (2, 2, 2), box, 1.5, 1.2 + 0.1j)
    assert abs(Db[1, 1, 1] - ((1 - (1.2 + 0.1j) / 1.5) + ((1.2 + 0.1j) / 1.5 - (1.2 + 0.1j) / (3.0 + 0.2j)) * 0.25)) <= 1e-15


def test_uniform_cell_closed_form_and_homogeneous_cell():
    """D = (1 - eps_b/eps_2) delta_d0, h perpendicular to k: H_0 = h (k_b^2 - kappa^2) / (k_b^2 - kappa^2 eps_b/eps_2)."""
    eps2, eps_b = 2.5, 1.3
    geo = wl.Geometry("u", (0.2, 0.2, 0.2), (3, 3, 3),
                      [dict(kind=wl.BOX, center=(0, 0, 0), size=(0.2, 0.2, 0.2), eps=eps2)], 1.0, eps_b, None, ())
    k0, kap = TWO_PI, 1.3 * TWO_PI
    H = orc.solve_dense_H(D_of(geo), geo.periods, geo.orders, np.array([0, 0, kap]), k0, eps_b, [0, 1.0, 0])
    kb2 = k0**2 * eps_b
    assert abs(orc.zero_order(H)[1] - (kb2 - kap**2) / (kb2 - kap**2 * eps_b / eps2)) <= 1e-13
    H[:, 1, 1, 1] = 0
    assert np.abs(H).max() <= 1e-14                                   # only m = 0 is excited
    hom = wl.sphere_lattice((3, 3, 3), eps=1.0)
    pol = np.array([0.3 - 0.2j, 1.0, 0.0])
    H = orc.solve_dense_H(D_of(hom), hom.periods, hom.orders, np.array([0, 0, kap]), k0, 1.0, pol)
    assert np.abs(H - orc.incident(hom.orders, pol)).max() <= 1e-15


def test_levi_civita_matrix_equals_cross_product_operator_and_gmres_equals_lu():
    geo = wl.Geometry("mix", (0.2, 0.25, 0.3), (3, 2, 4), wl.ellipsoid_lattice().shapes, 1.5, 1.3 + 0.1j, None, ())
    D = D_of(geo)
    kb, k0 = np.array([0.4, -0.3, 1.4 * TWO_PI]), 0.9 * TWO_PI
    x = wl.random_field(1, geo.orders, 3)[0]
    A = orc.assemble_dense_H(D, geo.periods, geo.orders, kb, k0, geo.eps_b)
    y = orc.apply_operator_H(D, x, geo.periods, kb, k0, geo.eps_b)
    assert np.abs((A @ x.ravel()).reshape(x.shape) - y).max() <= 1e-13 * np.abs(y).max()
    pol = [1.0, 0.5j, 0.0]
    H_lu = orc.solve_dense_H(D, geo.periods, geo.orders, kb, k0, geo.eps_b, pol)
    H_it, hist, _ = orc.solve_gmres_H(D, geo.periods, geo.orders, kb, k0, geo.eps_b, pol, tol=1e-13)
    assert np.linalg.norm(H_it - H_lu) <= 1e-11 * np.linalg.norm(H_lu) and np.all(np.diff(hist) <= 1e-15)


def test_solution_is_transverse():
    """Eq. 5 adds only vectors k_m x (...) to H^inc: k_m . H_m = 0 for every m when h is perpendicular to k_inc."""
    geo = wl.sphere_lattice((5, 5, 5))
    kinc = np.array([0.0, 0.0, 1.2 * TWO_PI])
    H = orc.solve_dense_H(D_of(geo), geo.periods, geo.orders, kinc, TWO_PI, geo.eps_b, [0, 1.0, 0])
    k = orc.wavevectors(geo.periods, geo.orders, kinc)
    assert np.abs((k * H).sum(axis=0)).max() <= 1e-13 * np.abs(H).max() * np.abs(k).max()


def _pole(geo, D, n_lo, n_hi, npts, axis=2, pol=(0, 1.0, 0), k0=TWO_PI):
    kappa = np.linspace(n_lo, n_hi, npts) * k0
    xi = np.zeros(npts, dtype=complex)
    pa = int(np.argmax(np.abs(pol)))
    for i, kv in enumerate(kappa):
        kinc = np.zeros(3); kinc[axis] = kv
        xi[i] = orc.zero_order(orc.solve_dense_H(D, geo.periods, geo.orders, kinc, k0, geo.eps_b, pol))[pa]
    eta, zeta = orc.pole_search(kappa, xi, 5, 10)
    b = orc.select_pole(eta, zeta, kappa[0], kappa[-1])
    assert b >= 0
    return eta[b]


def test_pole_is_an_eigenvalue_of_the_hermitian_plane_wave_operator():
    """Multiplying Eq. 5 by (k_b^2 - k_m^2) and using k.H = 0 gives  k0^2 H_m + k_m x sum [1/eps]_{m-m'} (k_m' x H_m')
    = source: at a pole, k0^2 is an eigenvalue of the Hermitian matrix Theta = -[k x][1/eps][k x] (the textbook
    H-field plane-wave expansion), independent of eps_b."""
    geo = wl.sphere_lattice((3, 3, 3))
    for eps_b in (1.0, 1.7):
        D = orc.coeffs_inverse_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, eps_b)
        g2 = wl.Geometry(geo.name, geo.periods, geo.orders, geo.shapes, geo.eps_bg, eps_b, None, ())
        eta = _pole(g2, D, 1.03, 1.17, 16)
        n = 27
        i = np.arange(3)
        i1, i2, i3 = [a.ravel() for a in np.meshgrid(i, i, i, indexing="ij")]
        inv_eps = -D / eps_b
        inv_eps[2, 2, 2] += 1.0 / eps_b                               # [1/eps]_d = (delta_d0 - D_d) / eps_b
        T = inv_eps[i1[:, None] - i1[None, :] + 2, i2[:, None] - i2[None, :] + 2, i3[:, None] - i3[None, :] + 2]
        k = orc.wavevectors(geo.periods, geo.orders, np.array([0, 0, eta.real])).reshape(3, n)

        def crossmat(kv):                                            # [3n x 3n] matrix of F -> k_m x F_m
            M = np.zeros((3 * n, 3 * n))
            for a, b, c in ((0, 1, 2), (1, 2, 0), (2, 0, 1)):
                M[a * n:(a + 1) * n, c * n:(c + 1) * n] += np.diag(kv[b])
                M[a * n:(a + 1) * n, b * n:(b + 1) * n] -= np.diag(kv[c])
            return M
        C = crossmat(k)
        Theta = -C @ np.kron(np.eye(3), T) @ C
        assert np.abs(Theta - Theta.conj().T).max() <= 1e-9 * np.abs(Theta).max()
        w = np.linalg.eigvalsh(0.5 * (Theta + Theta.conj().T))
        assert np.min(np.abs(w - TWO_PI**2)) / TWO_PI**2 <= 1e-7
        assert abs(eta.imag) <= 1e-8 * abs(eta.real)


def test_laminate_normal_incidence_converges_to_rytov_as_one_over_N():
    """k || z through the 1/9 laminate: the Laurent rule on [1/eps] d/dz converges only as ~1/N (PAPER.md:60, :123:
    the H-form is the less accurate one), but it converges to the Rytov root."""
    k0 = TWO_PI * 0.25 * 12 / 64
    k1, k2 = k0 * 1.0, k0 * 3.0
    cosK = np.cos(0.5 * k1) * np.cos(0.5 * k2) - 0.5 * (k1 / k2 + k2 / k1) * np.sin(0.5 * k1) * np.sin(0.5 * k2)
    n_rytov = np.arccos(cosK) / k0
    errs = []
    for N in (15, 31, 63):
        geo = wl.laminate((1, 1, N))
        eta = _pole(geo, D_of(geo), n_rytov * 0.93, n_rytov * 1.07, 16, axis=2, pol=(1.0, 0, 0), k0=k0)
        errs.append(abs(eta.real / k0 - n_rytov))
    assert errs[0] > errs[1] > errs[2] and errs[2] <= 2e-2
    assert 1.5 <= errs[0] / errs[1] <= 3.0 and 1.5 <= errs[1] / errs[2] <= 3.0      # ~1/N
