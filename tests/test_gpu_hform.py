"""GPU parity of the H-field formulation (Eq. 5; gsm.FORM_H) against the CPU oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

from oracle import gsm_oracle as orc  # noqa: E402
from paper_1501_01752_b200 import gsm, workloads as wl  # noqa: E402

TWO_PI = 2.0 * np.pi


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def D_of(geo):
    if geo.voxels is not None:
        return orc.coeffs_inverse_voxel(geo.voxels, geo.orders, geo.eps_b)
    return orc.coeffs_inverse_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)


def geometries():
    off = [dict(kind=wl.ELLIPSOID, center=(0.03, -0.02, 0.05), size=(0.04, 0.03, 0.04), eps=12.0 + 0.5j),
           dict(kind=wl.BOX, center=(-0.06, 0.07, 0.0), size=(0.04, 0.06, 0.3), eps=2.5)]
    rng = np.random.default_rng(wl.SEED)
    grid = (1.0 + 9.0 * rng.random((16, 8, 32))) + 0.3j * rng.random((16, 8, 32))
    return [wl.sphere_lattice((7, 7, 7)), wl.laminate((1, 1, 63)),
            wl.Geometry("mixed-even", (0.2, 0.25, 0.3), (5, 4, 6), off, 1.5, 1.3 + 0.1j, None, ()),
            wl.Geometry("vox", (0.2, 0.3, 0.25), (5, 3, 7), [], 1.0, 1.2, grid, ()),
            wl.Geometry("p64", (0.2, 0.25, 0.3), (17, 32, 25), wl.ellipsoid_lattice().shapes, 1.0, 1.1 + 0.05j, None, ())]


@pytest.mark.parametrize("geo", geometries(), ids=lambda g: g.name + "x".join(map(str, g.orders)))
def test_hform_coefficients_and_apply(geo):
    plan = gsm.plan_from_geometry(geo, max_batch=2, formulation=gsm.FORM_H)
    D = D_of(geo)
    assert np.max(np.abs(plan.coeffs() - D)) <= 1e-13 * max(1.0, np.max(np.abs(D)))
    x = wl.random_field(2, geo.orders, 21)
    rng = np.random.default_rng(22)
    kb = rng.uniform(-1.0, 1.0, (2, 3)) * TWO_PI * 1.3
    k0 = TWO_PI * rng.uniform(0.5, 1.5, 2)
    y = plan.apply(kb, k0, torch.from_numpy(x).cuda()).cpu().numpy()
    mv = orc.toeplitz_matvec_c if geo.n > 2000 else orc.toeplitz_matvec
    for b in range(2):
        ref = orc.apply_operator_H(D, x[b], geo.periods, kb[b], k0[b], geo.eps_b, mv)
        assert rel(y[b], ref) <= 1e-12
    plan.close()


def test_hform_apply_31cubed_sampled_rows():
    geo = wl.woodpile((31, 31, 31))
    plan = gsm.plan_from_geometry(geo, max_batch=1, formulation=gsm.FORM_H)
    D = D_of(geo)
    x = wl.random_field(1, geo.orders, 4)[0]
    kb, k0 = np.array([0.3, -0.2, 1.3 * TWO_PI]), TWO_PI
    y = plan.apply(kb[None], [k0], torch.from_numpy(x[None]).cuda()).cpu().numpy()[0]
    k = orc.wavevectors(geo.periods, geo.orders, kb)
    t = orc.cross_k(k, x)
    rng = np.random.default_rng(5)
    scale = np.sqrt(np.mean(np.abs(y) ** 2))
    for s in [(0, 0, 0), (30, 30, 30), (15, 15, 15)] + [tuple(int(v) for v in rng.integers(0, 31, 3)) for _ in range(12)]:
        F = orc.toeplitz_row(D, t, s)
        km = k[(slice(None),) + s]
        ref = x[(slice(None),) + s] - np.cross(km, F) / (k0**2 * geo.eps_b - np.dot(km, km))
        assert np.max(np.abs(y[(slice(None),) + s] - ref)) <= 1e-12 * scale
    plan.close()


def test_hform_solve_vs_dense_lu_and_transversality():
    geo = wl.sphere_lattice((7, 7, 7))
    plan = gsm.plan_from_geometry(geo, max_iters=100, formulation=gsm.FORM_H)
    kb, k0, pol = np.array([0.0, 0.0, 1.2 * TWO_PI]), TWO_PI, np.array([0.0, 1.0, 0.0], dtype=complex)
    H, hist, iters, resid, st = plan.solve(kb, k0, pol, tol=1e-12)
    ref = orc.solve_dense_H(D_of(geo), geo.periods, geo.orders, kb, k0, geo.eps_b, pol)
    Hn = H.cpu().numpy()
    assert st == gsm.OK and resid <= 1e-10 and rel(Hn, ref) <= 1e-9
    k = orc.wavevectors(geo.periods, geo.orders, kb)
    assert np.abs((k * Hn).sum(axis=0)).max() <= 1e-10 * np.abs(Hn).max() * np.abs(k).max()
    plan.close()


def test_hform_uniform_cell_closed_form():
    eps2, eps_b = 2.5, 1.3
    geo = wl.Geometry("u", (0.2, 0.2, 0.2), (3, 3, 3),
                      [dict(kind=wl.BOX, center=(0, 0, 0), size=(0.2, 0.2, 0.2), eps=eps2)], 1.0, eps_b, None, ())
    plan = gsm.plan_from_geometry(geo, formulation=gsm.FORM_H)
    k0, kap = TWO_PI, 1.3 * TWO_PI
    H, _, _, _, _ = plan.solve([0, 0, kap], k0, [0, 1.0, 0], tol=1e-13)
    kb2 = k0**2 * eps_b
    assert abs(orc.zero_order(H.cpu().numpy())[1] - (kb2 - kap**2) / (kb2 - kap**2 * eps_b / eps2)) <= 1e-12
    plan.close()


def test_hform_scan_pole_vs_oracle():
    """Scan + pole search in the H formulation (7^3 sphere lattice): eps_eff from both sides within 1e-8."""
    geo = wl.sphere_lattice((5, 5, 5))
    D = D_of(geo)
    kappa = wl.kappa_mesh(1.04, 1.16, 17)
    kb, kk, pol = wl.scan_points(kappa, 2, 1)
    plan = gsm.plan_from_geometry(geo, max_iters=100, max_batch=17, formulation=gsm.FORM_H)
    resp, iters, resid, st = plan.scan(kb, kk, pol, tol=1e-12)
    assert st == gsm.OK and np.all(resid <= 1e-10)
    xi = np.array([orc.zero_order(orc.solve_dense_H(D, geo.periods, geo.orders, kb[p], TWO_PI, geo.eps_b, [0, 1.0, 0]))[1]
                   for p in range(len(kappa))])
    assert np.max(np.abs(resp[:, 1] - xi) / np.abs(xi)) <= 1e-8
    eta, zeta, best = gsm.pole_search(kappa, resp[:, 1], 5, 10)
    eo, zo = orc.pole_search(kappa, xi, 5, 10)
    bo = orc.select_pole(eo, zo, kappa[0], kappa[-1])
    assert best >= 0 and bo >= 0 and abs((eta[best] / TWO_PI) ** 2 - (eo[bo] / TWO_PI) ** 2) <= 1e-8
    plan.close()
