"""Thin ctypes binding of the C ABI in include/gsm.h (argument marshalling only).

Every step of the hot path runs in the CUDA library ``libgsm_b200.so``; PyTorch is used for device memory and
the stream.  Importing this module fails loudly if the library has not been built - there is no CPU fallback.
Names follow include/gsm.h: Plan.apply / solve / scan and pole_search map 1:1 to gsm_apply / gsm_solve /
gsm_scan / gsm_pole_search.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgsm_b200.so")

OK, NOT_CONVERGED, E_INVALID, E_ALLOC, E_CUDA, E_SINGULAR_BASIS = 0, 1, -1, -2, -3, -4
SPHERE, ELLIPSOID, BOX, POLYHEDRON = 0, 1, 2, 3
FORM_E, FORM_H = 0, 1
FLAG_TWO_SWEEP, FLAG_GENERIC_APPLY, FLAG_FUSED_APPLY, FLAG_SLOT_REFILL = 1, 2, 4, 8   # include/gsm.h GSM_FLAG_*
MAX_ITERS = 512
STATIC_MAX_ORDER, STATIC_MAX_BATCH, STATIC_SCRATCH_BYTES = 16, 4, 2622720   # include/gsm.h GSM_STATIC_*


class GsmError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"gsm status {status}: {msg}")
        self.status = status


class _Shape(C.Structure):
    _fields_ = [("kind", C.c_int), ("center", C.c_double * 3), ("size", C.c_double * 3),
                ("eps_re", C.c_double), ("eps_im", C.c_double),
                ("n_vertices", C.c_int), ("vertices", C.c_void_p), ("n_faces", C.c_int), ("face_sizes", C.c_void_p),
                ("face_vertices", C.c_void_p)]


class _PlanDesc(C.Structure):
    _fields_ = [("period", C.c_double * 3), ("orders", C.c_int * 3),
                ("eps_bg_re", C.c_double), ("eps_bg_im", C.c_double),
                ("eps_b_re", C.c_double), ("eps_b_im", C.c_double),
                ("n_shapes", C.c_int), ("shapes", C.POINTER(_Shape)),
                ("voxels", C.c_int * 3), ("eps_grid_host", C.c_void_p),
                ("max_iters", C.c_int), ("max_batch", C.c_int), ("cuda_stream", C.c_void_p),
                ("formulation", C.c_int), ("flags", C.c_int)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'`. "
                          "There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    P = C.c_void_p
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int)
    lib.gsm_plan_create.argtypes = [C.POINTER(_PlanDesc), C.POINTER(P)]
    lib.gsm_plan_destroy.argtypes = [P]
    lib.gsm_plan_coeffs.argtypes = [P, P]
    lib.gsm_plan_info.argtypes = [P, ip, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    lib.gsm_apply.argtypes = [P, C.c_int, P, P, P, P]
    lib.gsm_solve.argtypes = [P, P, C.c_double, P, C.c_double, P, P, C.c_int, ip, dp]
    lib.gsm_plan_history.argtypes = [P, C.c_int, P, C.c_int, ip]
    lib.gsm_plan_history.restype = C.c_int
    lib.gsm_scan.argtypes = [P, C.c_int, P, P, P, C.c_double, P, P, P, P]
    lib.gsm_scan_guess.argtypes = [P, C.c_int, P, P, P, C.c_double, P, P, P, P, P]
    lib.gsm_scan_mesh.argtypes = [P, C.c_int, P, P, P, C.c_double, C.c_int, P, P, P, P]
    lib.gsm_mesh_schedule.argtypes = [C.c_int, C.c_int, C.c_int, P, P, P]
    lib.gsm_mesh_schedule.restype = C.c_int
    lib.gsm_pole_search.argtypes = [C.c_int, P, P, C.c_int, C.c_int, C.c_double, C.c_double, P, P, ip]
    lib.gsm_plan_set_cell.argtypes = [P, C.POINTER(_PlanDesc)]
    lib.gsm_plan_profile.argtypes = [P, C.c_int]
    lib.gsm_plan_profile_read.argtypes = [P, C.c_int, C.POINTER(C.c_longlong), dp, dp, C.c_int]
    lib.gsm_kernel_class_count.argtypes = []
    lib.gsm_kernel_class_count.restype = C.c_int
    lib.gsm_kernel_class_name.argtypes = [C.c_int]
    lib.gsm_kernel_class_name.restype = C.c_char_p
    lib.gsm_retrieve_neff.argtypes = [P, P, P, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double,
                                      C.c_double, P]
    lib.gsm_retrieve_neff.restype = C.c_int
    lib.gsm_retrieve_neff_many.argtypes = [P, C.c_int, P, P, P, P, P, P, C.c_int, C.c_int, C.c_double, C.c_double, P, P]
    lib.gsm_retrieve_neff_many.restype = C.c_int
    lib.gsm_apply_static.argtypes = [P, P, C.c_double, C.c_double, C.c_int, P, C.c_int, P, P, P, P, P]
    lib.gsm_apply_static.restype = C.c_int
    lib.gsm_last_error.argtypes = [P]
    lib.gsm_last_error.restype = C.c_char_p
    for f in ("gsm_plan_create", "gsm_plan_destroy", "gsm_plan_coeffs", "gsm_plan_info", "gsm_apply", "gsm_solve",
              "gsm_scan", "gsm_scan_guess", "gsm_scan_mesh", "gsm_pole_search", "gsm_plan_set_cell", "gsm_plan_profile",
              "gsm_plan_profile_read"):
        getattr(lib, f).restype = C.c_int
    return lib


_lib = _load()


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _check(status, plan=None, allow_warning=True):
    if status < 0 or (status > 0 and not allow_warning):
        raise GsmError(status, _lib.gsm_last_error(plan).decode())
    return status


class Plan:
    """gsm_plan: one periodic cell (periods, orders, shapes or voxel grid) on the current CUDA device."""

    def __init__(self, periods, orders, shapes=None, eps_bg=1.0, eps_b=None, voxels=None, max_iters=64, max_batch=1,
                 stream=None, formulation=FORM_E, flags=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1501_01752_b200.gsm needs a CUDA device; there is no CPU fallback")
        self._torch = torch
        self.stream = stream
        self.formulation = int(formulation)
        self.flags = int(flags)
        self.orders = tuple(int(n) for n in orders)
        d, keep = self._desc(periods, shapes, eps_bg, eps_b, voxels, max_iters, max_batch)
        self.n = int(np.prod(self.orders))
        self.max_batch, self.max_iters = int(max_batch), int(max_iters)
        self._keep = [keep]
        h = C.c_void_p()
        st = _lib.gsm_plan_create(C.byref(d), C.byref(h))
        if st != OK:
            raise GsmError(st, _lib.gsm_last_error(None).decode())
        self._h = h

    def _desc(self, periods, shapes, eps_bg, eps_b, voxels, max_iters, max_batch):
        """Marshal a gsm_plan_desc; `voxels` may be a complex128 numpy array or a (pinned) CPU torch tensor."""
        eps_b = eps_bg if eps_b is None else eps_b
        d = _PlanDesc()
        d.period[:] = [float(p) for p in periods]
        d.orders[:] = list(self.orders)
        d.eps_bg_re, d.eps_bg_im = complex(eps_bg).real, complex(eps_bg).imag
        d.eps_b_re, d.eps_b_im = complex(eps_b).real, complex(eps_b).imag
        if voxels is not None:
            if hasattr(voxels, "data_ptr"):          # torch CPU tensor (e.g. pinned), complex128, contiguous
                assert not voxels.is_cuda and voxels.is_contiguous() and voxels.dtype == self._torch.complex128
                grid, ptr = voxels, voxels.data_ptr()
            else:
                grid = np.ascontiguousarray(voxels, dtype=np.complex128)
                ptr = grid.ctypes.data
            d.voxels[:] = list(grid.shape)
            d.eps_grid_host = ptr
            d.n_shapes = 0
            keep = grid
        else:
            shapes = shapes or []
            arr = (_Shape * max(len(shapes), 1))()
            keep = [arr]
            for i, s in enumerate(shapes):
                arr[i].kind = int(s["kind"])
                arr[i].center[:] = [float(v) for v in s["center"]]
                arr[i].size[:] = [float(v) for v in s["size"]]
                arr[i].eps_re, arr[i].eps_im = complex(s["eps"]).real, complex(s["eps"]).imag
                if arr[i].kind == POLYHEDRON:
                    v = np.ascontiguousarray(s["vertices"], dtype=np.float64).reshape(-1, 3)
                    fs = np.ascontiguousarray([len(f) for f in s["faces"]], dtype=np.int32)
                    fv = np.ascontiguousarray([k for f in s["faces"] for k in f], dtype=np.int32)
                    keep += [v, fs, fv]
                    arr[i].n_vertices, arr[i].vertices = len(v), v.ctypes.data
                    arr[i].n_faces, arr[i].face_sizes, arr[i].face_vertices = len(fs), fs.ctypes.data, fv.ctypes.data
            d.n_shapes = len(shapes)
            d.shapes = arr
            d.voxels[:] = [0, 0, 0]
            d.eps_grid_host = None
        d.max_iters, d.max_batch = int(max_iters), int(max_batch)
        d.cuda_stream = self.stream.cuda_stream if self.stream is not None else None
        d.formulation = self.formulation
        d.flags = self.flags
        return d, keep

    def set_cell(self, periods, shapes=None, eps_bg=1.0, eps_b=None, voxels=None):
        """gsm_plan_set_cell: re-run step a0 for a new cell with the same orders, keeping all workspaces."""
        d, keep = self._desc(periods, shapes, eps_bg, eps_b, voxels, self.max_iters, self.max_batch)
        _check(_lib.gsm_plan_set_cell(self._h, C.byref(d)), self._h)
        del keep

    def profile(self, enable=True):
        """gsm_plan_profile: bracket every kernel launch with CUDA events on the plan's stream."""
        _check(_lib.gsm_plan_profile(self._h, 1 if enable else 0), self._h)

    def profile_read(self, reset=False):
        """gsm_plan_profile_read: {class name: (launches, total ms, algorithmic bytes)}."""
        n = _lib.gsm_kernel_class_count()
        cnt = (C.c_longlong * n)()
        ms = (C.c_double * n)()
        by = (C.c_double * n)()
        _check(_lib.gsm_plan_profile_read(self._h, n, cnt, ms, by, 1 if reset else 0), self._h)
        return {_lib.gsm_kernel_class_name(c).decode(): (int(cnt[c]), float(ms[c]), float(by[c])) for c in range(n)}

    # -- lifetime -------------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            _lib.gsm_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- queries --------------------------------------------------------------------------------------------
    def coeffs(self) -> np.ndarray:
        N = self.orders
        out = np.empty((2 * N[0] - 1, 2 * N[1] - 1, 2 * N[2] - 1), dtype=np.complex128)
        _check(_lib.gsm_plan_coeffs(self._h, out.ctypes.data), self._h)
        return out

    def info(self):
        g = (C.c_int * 3)()
        b, l = C.c_longlong(), C.c_longlong()
        _check(_lib.gsm_plan_info(self._h, g, C.byref(b), C.byref(l)), self._h)
        return {"fft_grid": tuple(g), "device_bytes": b.value, "launches": l.value}

    # -- hot path -------------------------------------------------------------------------------------------
    def _order_before(self):
        """Plan bound to a side stream: make it wait for the work already queued on torch's current stream (which may
        still be producing the tensors handed in).  Returns the current stream, or None when no ordering is needed."""
        cur = self._torch.cuda.current_stream()
        if self.stream is None or self.stream == cur:
            return None
        self.stream.wait_stream(cur)
        return cur

    def _order_after(self, cur, *tensors):
        """Counterpart of _order_before: the current stream waits for the plan's stream, and the caching allocator is
        told that the plan's stream used `tensors` (so their memory is not recycled under it)."""
        if cur is None:
            return
        cur.wait_stream(self.stream)
        for t in tensors:
            if t is not None:
                t.record_stream(self.stream)

    def apply(self, k_bloch, k0, x, out=None):
        """gsm_apply: y = x - G (T x).  x: cuda complex128 tensor [batch, 3, N1, N2, N3].

        Asynchronous on the plan's stream; ordered after the work already queued on torch's current stream (which
        produced x) and before whatever the current stream does next (which may read y)."""
        torch = self._torch
        batch = x.shape[0]
        assert x.is_cuda and x.dtype == torch.complex128 and x.is_contiguous() and tuple(x.shape[1:]) == (3,) + self.orders
        y = torch.empty_like(x) if out is None else out
        kb, kk = _f64(k_bloch, (batch, 3)), _f64(k0, (batch,))
        cur = self._order_before()
        try:
            _check(_lib.gsm_apply(self._h, batch, kb.ctypes.data, kk.ctypes.data, x.data_ptr(), y.data_ptr()), self._h)
        finally:
            self._order_after(cur, x, y)
        return y

    def solve(self, k_bloch, k0, pol, tol=1e-10, out=None):
        """gsm_solve: returns (E cuda tensor [3,N1,N2,N3], residual history, iterations, true residual, status).
        Ordered against torch's current stream like apply()."""
        torch = self._torch
        E = torch.empty((3,) + self.orders, dtype=torch.complex128, device="cuda") if out is None else out
        kb = _f64(k_bloch, (3,))
        pl = _f64(np.asarray(pol, dtype=np.complex128).view(np.float64), (6,))
        hist = np.zeros(self.max_iters)
        it, res = C.c_int(), C.c_double()
        cur = self._order_before()
        try:
            st = _check(_lib.gsm_solve(self._h, kb.ctypes.data, float(k0), pl.ctypes.data, float(tol), E.data_ptr(),
                                       hist.ctypes.data, self.max_iters, C.byref(it), C.byref(res)), self._h)
        finally:
            self._order_after(cur, E)
        return E, hist[: it.value].copy(), it.value, res.value, st

    def history(self, b=0):
        """gsm_plan_history: residual estimates of solve b of the most recent lock-step batch."""
        hist = np.zeros(self.max_iters)
        it = C.c_int()
        _check(_lib.gsm_plan_history(self._h, int(b), hist.ctypes.data, self.max_iters, C.byref(it)), self._h)
        return hist[: it.value].copy()

    def scan(self, k_bloch, k0, pol, tol=1e-10, fields=None, x0=None, levels=None):
        """gsm_scan: returns (resp [npts,3] complex, iters [npts], resid [npts], status).

        pol: [npts, 6] real (interleaved complex) or [npts, 3] complex.  fields: optional cuda tensor
        [npts, 3, N1, N2, N3] that receives every solution.  x0: optional cuda tensor of the same shape with initial
        guesses (gsm_scan_guess; may be `fields` itself).  levels: solve the list as an ordered equidistant mesh in
        that many coarse-to-fine waves, each started from the interpolation of the previous ones (gsm_scan_mesh).
        With the plan on a side stream the call is ordered after torch's current stream (which may still be writing x0)
        and the current stream after the call (which may read fields), like apply()."""
        kb = _f64(k_bloch)
        npts = kb.shape[0]
        kk = _f64(k0, (npts,))
        pl = np.asarray(pol)
        if np.iscomplexobj(pl):
            pl = np.ascontiguousarray(pl, dtype=np.complex128).view(np.float64)
        pl = _f64(pl, (npts, 6))
        resp = np.zeros((npts, 3), dtype=np.complex128)
        iters = np.zeros(npts, dtype=np.int32)
        resid = np.zeros(npts)
        fp = fields.data_ptr() if fields is not None else None
        cur = self._order_before()
        try:
            st = self._scan_call(npts, kb, kk, pl, tol, levels, x0, resp, iters, resid, fp)
        finally:
            self._order_after(cur, x0, fields)
        return resp, iters, resid, _check(st, self._h)

    def _scan_call(self, npts, kb, kk, pl, tol, levels, x0, resp, iters, resid, fp):
        if levels is not None:
            assert x0 is None
            st = _lib.gsm_scan_mesh(self._h, npts, kb.ctypes.data, kk.ctypes.data, pl.ctypes.data, float(tol), int(levels),
                                    resp.ctypes.data, iters.ctypes.data, resid.ctypes.data, fp)
        elif x0 is not None:
            assert x0.is_cuda and x0.is_contiguous() and tuple(x0.shape) == (npts, 3) + self.orders
            st = _lib.gsm_scan_guess(self._h, npts, kb.ctypes.data, kk.ctypes.data, pl.ctypes.data, float(tol),
                                     x0.data_ptr(), resp.ctypes.data, iters.ctypes.data, resid.ctypes.data, fp)
        else:
            st = _lib.gsm_scan(self._h, npts, kb.ctypes.data, kk.ctypes.data, pl.ctypes.data, float(tol),
                               resp.ctypes.data, iters.ctypes.data, resid.ctypes.data, fp)
        return st


    def retrieve_neff(self, direction, pol, comp, k0, n_lo, n_hi, ncoarse=29, nfine=18, fine_step=0.002, tol=1e-10):
        """gsm_retrieve_neff: returns (n_eff, eps_eff, zeta, status) for one (direction, polarisation) pair."""
        d = _f64(direction, (3,))
        pl = _f64(np.asarray(pol, dtype=np.complex128).view(np.float64), (6,))
        out = np.zeros(6)
        st = _check(_lib.gsm_retrieve_neff(self._h, d.ctypes.data, pl.ctypes.data, int(comp), float(k0), float(n_lo),
                                           float(n_hi), int(ncoarse), int(nfine), float(fine_step), float(tol),
                                           out.ctypes.data), self._h)
        return complex(out[0], out[1]), complex(out[2], out[3]), complex(out[4], out[5]), st


    def retrieve_neff_many(self, directions, pols, comps, k0, n_lo, n_hi, ncoarse=29, nfine=18, fine_step=0.002, tol=1e-10):
        """gsm_retrieve_neff_many: nlines retrievals with every stage in one scan.  directions [n,3]; pols [n,3] complex;
        comps [n] (component index, or -1 = projection on the amplitude); k0, n_lo, n_hi scalars or [n].
        Returns (n_eff [n] complex, eps_eff [n] complex, zeta [n] complex, line_status [n], status)."""
        d = _f64(directions)
        n = d.shape[0]
        pl = _f64(np.ascontiguousarray(pols, dtype=np.complex128).view(np.float64), (n, 6))
        cp = np.ascontiguousarray(np.broadcast_to(np.asarray(comps, dtype=np.int32), (n,)))
        kk, lo, hi = (_f64(np.broadcast_to(np.asarray(v, dtype=np.float64), (n,))) for v in (k0, n_lo, n_hi))
        out = np.zeros((n, 6))
        ls = np.full(n, E_INVALID, dtype=np.int32)
        st = _lib.gsm_retrieve_neff_many(self._h, n, d.ctypes.data, pl.ctypes.data, cp.ctypes.data, kk.ctypes.data,
                                         lo.ctypes.data, hi.ctypes.data, int(ncoarse), int(nfine), float(fine_step),
                                         float(tol), out.ctypes.data, ls.ctypes.data)
        if st < 0 and not np.any(ls == OK):
            _check(st, self._h)
        return out[:, 0] + 1j * out[:, 1], out[:, 2] + 1j * out[:, 3], out[:, 4] + 1j * out[:, 5], ls, st


def apply_static(periods, orders, eps_b, coef, k_bloch, k0, x, out, formulation=FORM_E, stream=None):
    """gsm_apply_static: y = x - G (T x) without a plan, for programs that must not touch the CUDA allocator.

    Meant for hosts whose own allocator already owns the GPU's memory (or that run under a memory quota, or cannot
    afford cudaMalloc's device-wide synchronisation): the library allocates nothing here, its intermediates live in a
    fixed STATIC_SCRATCH_BYTES array inside the library image.  In the same spirit this wrapper allocates nothing on the
    device either - `out` is required.  coef: cuda complex128 tensor [2N1-1, 2N2-1, 2N3-1] (layout of Plan.coeffs());
    x, out: cuda complex128 [batch, 3, N1, N2, N3], distinct; orders <= STATIC_MAX_ORDER per axis, batch <=
    STATIC_MAX_BATCH (larger sizes raise GsmError naming the limit).  Enqueued on `stream` (default: torch's current
    stream).  One scratch array per GPU is shared by all calls: do not let two calls overlap on the device."""
    import torch
    orders = tuple(int(n) for n in orders)
    batch = int(x.shape[0])
    for t in (coef, x, out):
        assert t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()
    assert tuple(coef.shape) == tuple(2 * n - 1 for n in orders)
    assert tuple(x.shape) == (batch, 3) + orders and tuple(out.shape) == tuple(x.shape)
    per = _f64(periods, (3,))
    od = np.ascontiguousarray(orders, dtype=np.int32)
    kb, kk = _f64(k_bloch, (batch, 3)), _f64(k0, (batch,))
    st = (stream if stream is not None else torch.cuda.current_stream()).cuda_stream
    _check(_lib.gsm_apply_static(per.ctypes.data, od.ctypes.data, complex(eps_b).real, complex(eps_b).imag, int(formulation),
                                 coef.data_ptr(), batch, kb.ctypes.data, kk.ctypes.data, x.data_ptr(), out.data_ptr(), st))
    return out


def mesh_schedule(npts, levels, collapse_after=0):
    """gsm_mesh_schedule (host side): (wave [npts], nodes [npts, 8], weights [npts, 8]) of gsm_scan_mesh."""
    wave = np.full(npts, -1, dtype=np.int32)
    nodes = np.full((npts, 8), -1, dtype=np.int32)
    weights = np.zeros((npts, 8))
    st = _lib.gsm_mesh_schedule(int(npts), int(levels), int(collapse_after), wave.ctypes.data, nodes.ctypes.data,
                                weights.ctypes.data)
    if st < 0:
        raise GsmError(st, "gsm_mesh_schedule: invalid arguments")
    return wave, nodes, weights


def pole_search(kappa, xi, Np=5, Nd=10, lo=None, hi=None):
    """gsm_pole_search (host side): returns (eta [Np], zeta [Np], best index or -1)."""
    kappa = _f64(kappa)
    xi = np.ascontiguousarray(xi, dtype=np.complex128)
    eta = np.zeros(Np, dtype=np.complex128)
    zeta = np.zeros(Np, dtype=np.complex128)
    best = C.c_int(-1)
    lo = float(kappa[0]) if lo is None else float(lo)
    hi = float(kappa[-1]) if hi is None else float(hi)
    st = _lib.gsm_pole_search(len(kappa), kappa.ctypes.data, xi.ctypes.data, int(Np), int(Nd), lo, hi,
                              eta.ctypes.data, zeta.ctypes.data, C.byref(best))
    if st < 0:
        raise GsmError(st, "gsm_pole_search: invalid arguments")
    return eta, zeta, best.value


def plan_from_geometry(geo, max_iters=64, max_batch=1, stream=None, formulation=FORM_E, flags=0) -> Plan:
    """Plan for a workloads.Geometry (seeded input description; holds no arithmetic of the method)."""
    return Plan(geo.periods, geo.orders, shapes=geo.shapes, eps_bg=geo.eps_bg, eps_b=geo.eps_b, voxels=geo.voxels,
                max_iters=max_iters, max_batch=max_batch, stream=stream, formulation=formulation, flags=flags)
