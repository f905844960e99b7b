"""gsm_apply_static - the operator apply for programs that are not allowed to allocate GPU memory.

Some hosts of this library cannot call cudaMalloc: their own allocator (PyTorch's caching allocator, a serving
engine's pre-reserved pool) already owns the device, or they run under a memory quota, or they sit in a loop that
cannot take cudaMalloc's device-wide synchronisation.  A gsm_plan is out of reach for them (gsm_plan_create allocates),
so include/gsm.h offers ONE plan-free entry point whose intermediates live in a fixed array inside the library image.
These tests hold it to the plan-based path (gsm_apply) at the tolerance the other operator tests use (relative L2
<= 1e-12; the kernels are the same, so the results are normally identical), on consecutive calls that share the array:
a large call first, a smaller one after it, so that the second runs over the first one's left-overs.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here should not hide
the parity tests.  It must pass alone in a fresh process and after the other modules (the entry point sets itself up on
its first call per device, whenever that is).
"""
import ctypes

import numpy as np
import pytest

from paper_1501_01752_b200 import gsm, workloads as wl

TWO_PI = 2.0 * np.pi


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return torch


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def _case(torch, geo, batch, seed, formulation, y_static, poison):
    """One call of each path on the same inputs; returns (static result, plan result) as numpy arrays."""
    plan = gsm.plan_from_geometry(geo, max_batch=batch, formulation=formulation)
    coef = torch.from_numpy(plan.coeffs()).cuda()               # the generator c_d, now in a buffer the caller owns
    x = torch.from_numpy(wl.random_field(batch, geo.orders, seed)).cuda()
    rng = np.random.default_rng(seed + 1)
    kb = rng.uniform(-1.0, 1.0, (batch, 3)) * TWO_PI * 1.3
    k0 = TWO_PI * rng.uniform(0.5, 1.5, batch)
    y_plan = plan.apply(kb, k0, x)
    out = y_static[: x.numel()].view(x.shape)
    out.fill_(poison)                                            # a call that wrote nothing would be caught
    gsm.apply_static(geo.periods, geo.orders, geo.eps_b, coef, kb, k0, x, out, formulation=formulation)
    torch.cuda.synchronize()
    res = out.cpu().numpy().copy(), y_plan.cpu().numpy()
    plan.close()
    return res


@pytest.mark.gpu
def test_static_apply_matches_the_plan_path_on_consecutive_calls():
    torch = _cuda()
    big = wl.Geometry("static-max", (0.2, 0.25, 0.3), (16, 16, 16), wl.ellipsoid_lattice().shapes, 1.0, 1.1 + 0.05j, None, ())
    small = wl.Geometry("static-ragged", (0.2, 0.25, 0.3), (7, 5, 9), wl.ellipsoid_lattice().shapes, 1.5, 1.3 + 0.1j, None, ())
    flat = wl.sphere_lattice((7, 7, 7))
    # every output goes to one buffer allocated up front: between the calls below nothing new is needed for y
    y_static = torch.empty(gsm.STATIC_MAX_BATCH * 3 * 16 ** 3, dtype=torch.complex128, device="cuda")
    calls = [(big, gsm.STATIC_MAX_BATCH, 21, gsm.FORM_E),        # the maximum: fills the whole scratch array
             (small, 2, 22, gsm.FORM_E),                         # right after it, smaller and ragged: runs over left-overs
             (small, 3, 23, gsm.FORM_H),                         # Eq. 5 through the same entry point
             (flat, 1, 24, gsm.FORM_E)]
    for geo, batch, seed, form in calls:
        ys, yp = _case(torch, geo, batch, seed, form, y_static, complex(np.nan, np.nan))
        assert np.all(np.isfinite(ys.view(np.float64))), (geo.name, "output not fully written")
        assert rel(ys, yp) <= 1e-12, (geo.name, batch, form, rel(ys, yp))
    # the same call twice in a row gives the same bits (nothing left in the array leaks into the next result)
    a, _ = _case(torch, small, 2, 22, gsm.FORM_E, y_static, 0.0)
    b, _ = _case(torch, small, 2, 22, gsm.FORM_E, y_static, 0.0)
    assert np.array_equal(a.view(np.float64), b.view(np.float64))


@pytest.mark.gpu
def test_static_apply_against_the_oracle():
    """Independent of the plan path: the oracle's O(n^2) Toeplitz product and Green dyadic on the same inputs."""
    torch = _cuda()
    from oracle import gsm_oracle as orc
    geo = wl.sphere_lattice((7, 7, 7))
    c = orc.coeffs_analytic(geo.periods, geo.orders, geo.shapes, geo.eps_bg, geo.eps_b)
    x = wl.random_field(2, geo.orders, 31)
    kb = np.array([[0.3, -0.2, 1.2 * TWO_PI], [1.1 * TWO_PI, 0.0, 0.4]])
    k0 = np.array([TWO_PI, 0.8 * TWO_PI])
    out = torch.empty((2, 3) + tuple(geo.orders), dtype=torch.complex128, device="cuda")
    for _ in range(2):
        out.zero_()
        gsm.apply_static(geo.periods, geo.orders, geo.eps_b, torch.from_numpy(c).cuda(), kb, k0, torch.from_numpy(x).cuda(), out)
        y = out.cpu().numpy()
        for b in range(2):
            ref = orc.apply_operator(c, x[b], geo.periods, kb[b], k0[b], geo.eps_b)
            assert rel(y[b], ref) <= 1e-12


def test_static_apply_refuses_sizes_beyond_its_fixed_scratch():
    """Host-side validation only (runs without a GPU): too many orders or too large a batch is an error that names the
    limit, never a silent overrun of the fixed array."""
    lib = ctypes.CDLL(gsm.LIB_PATH)
    lib.gsm_apply_static.restype = ctypes.c_int
    lib.gsm_apply_static.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                     ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 5
    lib.gsm_last_error.restype = ctypes.c_char_p
    lib.gsm_last_error.argtypes = [ctypes.c_void_p]
    per = np.array([0.2, 0.2, 0.2])
    kb, k0 = np.zeros((8, 3)), np.full(8, TWO_PI)
    fake = 0x1000   # stands for device pointers; rejected calls never touch them

    def call(orders, batch, d_x=fake, d_y=2 * fake):
        od = np.array(orders, dtype=np.int32)
        return lib.gsm_apply_static(per.ctypes.data, od.ctypes.data, 1.0, 0.0, 0, fake, batch, kb.ctypes.data, k0.ctypes.data,
                                    d_x, d_y, None)

    assert call((gsm.STATIC_MAX_ORDER + 1, 3, 3), 1) == gsm.E_INVALID
    assert b"GSM_STATIC_MAX_ORDER" in lib.gsm_last_error(None)
    assert call((3, 3, gsm.STATIC_MAX_ORDER + 1), 1) == gsm.E_INVALID
    assert call((3, 3, 3), gsm.STATIC_MAX_BATCH + 1) == gsm.E_INVALID
    assert b"GSM_STATIC_MAX_BATCH" in lib.gsm_last_error(None)
    assert call((3, 3, 3), 0) == gsm.E_INVALID
    assert call((3, 3, 3), 1, d_x=fake, d_y=fake) == gsm.E_INVALID      # in place is not supported
    assert call((3, 0, 3), 1) == gsm.E_INVALID
