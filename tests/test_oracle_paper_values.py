"""The oracle against the numbers the paper prints (tests/golden/paper_values.txt; CPU only).

The printed effective indices are converged values; the truncated E-form approaches them as ~1/N (SURVEY 8(c)
P-table), so the check is the 1/N (Richardson) extrapolation from two truncations.  A convention error
(sign, units, factor 2 pi, wrong tensor slot) moves n_eff at the 1e-2 level and fails these.
"""
import numpy as np
import pytest

from conftest import load_golden
from oracle import gsm_oracle as O
from paper_1501_01752_b200 import workloads as W

K0 = 2 * np.pi
GOLD = load_golden()


def n_eff_truncated(kind, n_host, N, n_lo, n_hi):
    g = W.cavity_lattice((N, N, N), kind, n_host)
    c = O.coeffs_analytic(g.periods, g.orders, g.shapes, g.eps_bg, g.eps_b)
    kap = W.kappa_mesh(n_lo, n_hi, 16)
    xi, its = [], []
    for kp in kap:
        if N <= 7:
            E = O.solve_dense(c, g.periods, g.orders, np.array([0, 0, kp]), K0, g.eps_b, [1, 0, 0])
        else:
            E, _, m = O.solve_gmres(c, g.periods, g.orders, np.array([0, 0, kp]), K0, g.eps_b, [1, 0, 0],
                                    tol=1e-12, matvec=O.toeplitz_matvec_c)
            its.append(m)
        xi.append(O.zero_order(E)[0])
    eta, zeta = O.pole_search(kap, xi, 5, 10)
    j = O.select_pole(eta, zeta, kap[0], kap[-1])
    assert j >= 0 and abs(eta[j].imag) < 1e-7 * K0
    return eta[j].real / K0, its


@pytest.mark.parametrize("kind,n_host,key,window,tol", [
    ("sphere", 1.5, "n_eff_sphere_cavity_host_1.5", (1.33, 1.39), 1e-4),
    ("cube", 1.5, "n_eff_cube_cavity_host_1.5", (1.41, 1.47), 3e-4),
    ("sphere", 3.0, "n_eff_sphere_cavity_host_3.0", (2.50, 2.58), 5e-4),
    ("cube", 3.0, "n_eff_cube_cavity_host_3.0", (2.76, 2.88), 1e-3),      # sharp edges at high contrast: slowest 1/N tail
])
def test_printed_effective_index_by_1_over_N_extrapolation(kind, n_host, key, window, tol):
    n7, _ = n_eff_truncated(kind, n_host, 7, *window)
    n15, its = n_eff_truncated(kind, n_host, 15, *window)
    n_inf = n15 - (n7 - n15) * (1 / 15) / (1 / 7 - 1 / 15)
    assert abs(n_inf - GOLD[key]) < tol, (n7, n15, n_inf)
    assert abs(n15 - GOLD[key]) < abs(n7 - GOLD[key])
    # "about 10 for low-contrast ... about 50 for high-contrast"
    assert GOLD["gmres_iters_low"] - 4 <= min(its) and max(its) <= GOLD["gmres_iters_high"] + 15


def test_maxwell_garnett_values():
    """eps_MG = eps_h (1 + 3 f beta/(1 - f beta)), beta = (eps_i-eps_h)/(eps_i+2 eps_h) (textbook)."""
    eh, ei = 2.25, 1.0
    beta = (ei - eh) / (ei + 2 * eh)
    for f, key in [((4 / 3) * np.pi / 27, "n_mg_uniaxial"), ((4 / 3) * np.pi / 27 / 1.1, "n_mg_biaxial")]:
        n = np.sqrt(eh * (1 + 3 * f * beta / (1 - f * beta)))
        assert abs(n - GOLD[key]) < 6e-5
    # the GSM long-wavelength limit must approach MG from the rigorous side: period 0.03 lambda, 7^3 orders
    L = 0.03
    shapes = [dict(kind=W.SPHERE, center=(0, 0, 0), size=(L / 3, 0, 0), eps=1.0)]
    c = O.coeffs_analytic((L, L, L), (7, 7, 7), shapes, 2.25, 2.25)
    kap = W.kappa_mesh(1.40, 1.45, 16)
    xi = [O.zero_order(O.solve_dense(c, (L, L, L), (7, 7, 7), np.array([0, 0, kp]), K0, 2.25, [1, 0, 0]))[0] for kp in kap]
    eta, zeta = O.pole_search(kap, xi, 5, 10)
    j = O.select_pole(eta, zeta, kap[0], kap[-1])
    assert abs(eta[j].real / K0 - GOLD["n_mg_uniaxial"]) < 3e-3
