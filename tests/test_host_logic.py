"""CPU-only checks of the boundary and the host logic (no compute calls on a GPU):
  * the C-ABI library builds, loads and exports every symbol include/gsm.h declares;
  * gsm_pole_search (host code of the library) against the oracle's pole search and a synthetic meromorphic function;
  * the binding refuses to run without a CUDA device (no CPU fallback);
  * the multi-GPU scan sharding (scan_shard.py) with torch.distributed gloo, world_size 2.
"""
import ctypes
import os
import re
import socket

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1501_01752_b200.build import build_cuda
    return build_cuda()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gsm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gsm_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib_path):
    names = declared_functions()
    assert {"gsm_plan_create", "gsm_plan_destroy", "gsm_apply", "gsm_solve", "gsm_scan", "gsm_pole_search",
            "gsm_plan_set_cell", "gsm_plan_profile", "gsm_plan_profile_read", "gsm_last_error", "gsm_scan_guess",
            "gsm_scan_mesh", "gsm_retrieve_neff_many", "gsm_mesh_schedule", "gsm_plan_history"} <= set(names)
    lib = ctypes.CDLL(lib_path)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/gsm.h but not exported by {lib_path}"


def test_kernel_class_names(lib_path):
    lib = ctypes.CDLL(lib_path)
    lib.gsm_kernel_class_name.restype = ctypes.c_char_p
    n = lib.gsm_kernel_class_count()
    names = [lib.gsm_kernel_class_name(i).decode() for i in range(n)]
    assert len(set(names)) == n and "arnoldi_mgs" in names and "xy_conv" in names


def test_null_arguments_are_rejected_without_a_device(lib_path):
    lib = ctypes.CDLL(lib_path)
    out = ctypes.c_void_p()
    assert lib.gsm_plan_create(None, ctypes.byref(out)) == -1 and not out.value
    assert lib.gsm_plan_destroy(None) == -1
    assert lib.gsm_apply(None, 1, None, None, None, None) == -1


def test_binding_has_no_cpu_fallback():
    import torch
    from paper_1501_01752_b200 import gsm
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        gsm.Plan((1.0, 1.0, 1.0), (3, 3, 3))


@pytest.mark.parametrize("npts,levels,collapse", [(256, 5, 0), (256, 5, 1), (45, 4, 2), (45, 4, 0), (21, 3, 0), (9, 6, 1),
                                                  (2, 5, 0), (1, 3, 0), (1024, 7, 1), (100, 1, 0)])
def test_mesh_schedule_waves_and_stencils(npts, levels, collapse):
    """gsm_mesh_schedule = the host logic of gsm_scan_mesh (reading R25), no device needed: every point is solved exactly
    once; wave 0 is an equidistant subset holding the first point; a point's interpolation nodes were all solved in
    EARLIER waves, are distinct, and are the nearest solved points; the Lagrange weights sum to one and reproduce every
    polynomial of degree below the node count at the point's own index."""
    from paper_1501_01752_b200 import gsm
    wave, nodes, w = gsm.mesh_schedule(npts, levels, collapse)
    assert wave.min() == 0 and np.all(wave >= 0)
    if collapse > 0:
        assert wave.max() <= collapse + 1
    z = np.flatnonzero(wave == 0)
    assert z[0] == 0 and (len(z) == 1 or len(set(np.diff(z).tolist())) == 1)
    if npts >= 2:
        assert len(z) >= 2 or levels == 1 or npts == 2                 # levels were reduced to what the list supports
    if levels == 1:
        assert np.all(wave == 0) and np.all(nodes == -1)
    for p in range(npts):
        nd = nodes[p][nodes[p] >= 0]
        if wave[p] == 0:
            assert len(nd) == 0
            continue
        assert len(nd) >= 2 and len(set(nd.tolist())) == len(nd)
        assert np.all(wave[nd] < wave[p]) and np.all((nd >= 0) & (nd < npts))
        solved = np.flatnonzero(wave < wave[p])
        nearest = solved[np.argsort(np.abs(solved - p), kind="stable")[:len(nd)]]
        assert np.abs(nd - p).max() <= np.abs(nearest - p).max() + 2 * np.abs(nd - p).min()    # a compact neighbourhood
        wp = w[p][:len(nd)]
        assert abs(wp.sum() - 1.0) <= 1e-9
        t = (nd - p) / max(1.0, float(np.abs(nd - p).max()))           # scaled offsets: polynomials in t vanish-order test
        for deg in range(1, len(nd)):
            assert abs(np.dot(wp, t**deg)) <= 1e-8 * max(1.0, np.abs(wp).max()), (p, deg)
    with pytest.raises(gsm.GsmError):
        gsm.mesh_schedule(5, 0)


def test_pole_search_matches_oracle_and_synthetic_poles():
    from oracle import gsm_oracle as orc
    from paper_1501_01752_b200 import gsm
    kappa = np.linspace(6.8, 7.9, 21)
    eta_true = np.array([7.31 + 0.004j, 9.2 - 0.01j])
    zeta_true = np.array([0.37 - 0.11j, 0.05 + 0.02j])
    xi = sum(z / (kappa - e) for z, e in zip(zeta_true, eta_true)) + 0.3 - 0.02 * kappa + 0.004 * kappa**2
    eta, zeta, best = gsm.pole_search(kappa, xi, 5, 10)
    assert best >= 0
    assert abs(eta[best] - eta_true[0]) <= 1e-10 and abs(zeta[best] - zeta_true[0]) <= 1e-8
    eta_o, zeta_o = orc.pole_search(kappa, xi, 5, 10)
    bo = orc.select_pole(eta_o, zeta_o, kappa[0], kappa[-1])
    assert abs(eta[best] - eta_o[bo]) <= 1e-10 and abs(zeta[best] - zeta_o[bo]) <= 1e-8
    with pytest.raises(gsm.GsmError):
        gsm.pole_search(kappa[:8], xi[:8], 5, 10)          # fewer than Np + Nd points


# ------------------------------------------------------------------------------------------- scan sharding
def test_shard_bounds_partition():
    from paper_1501_01752_b200.scan_shard import shard_bounds
    for npts in (0, 1, 7, 256, 257):
        for world in (1, 2, 3, 8):
            blocks = [shard_bounds(npts, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == npts
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_bounds(4, 2, 2)


def _fake_scan(kb, k0, pol):
    """Stand-in for Plan.scan on CPU ranks: a deterministic function of each point (no method arithmetic)."""
    resp = np.stack([kb[:, 2] + 1j * k0, kb[:, 0] * 0 + pol[:, 0], 2.0 * kb[:, 2]], axis=1).astype(np.complex128)
    return resp, (kb[:, 2] * 10).astype(np.int32), 1e-12 * k0


def _gloo_worker(rank, world, port, npts, q):
    import torch.distributed as dist
    from paper_1501_01752_b200.scan_shard import sharded_scan
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    rng = np.random.default_rng(5)
    kb = rng.uniform(0, 9, (npts, 3)); k0 = rng.uniform(5, 7, npts); pol = rng.uniform(0, 1, (npts, 6))
    calls = []

    def scan_fn(a, b, c):
        calls.append(len(a))
        return _fake_scan(a, b, c)
    resp, iters, resid = sharded_scan(scan_fn, kb, k0, pol, rank, world)
    ref = _fake_scan(kb, k0, pol)
    ok = np.array_equal(resp, ref[0]) and np.array_equal(iters, ref[1]) and np.array_equal(resid, ref[2])
    q.put((rank, bool(ok), calls))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("npts", [9, 1])
def test_sharded_scan_gloo_world2(npts):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, npts, q)) for r in range(2)]
    for p in procs:
        p.start()
    results = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in results)
    sizes = {r: sum(c) for r, _, c in results}
    assert sizes[0] + sizes[1] == npts and abs(sizes[0] - sizes[1]) <= 1
