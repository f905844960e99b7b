"""CPU oracle for the 3-D Generalized Source Method (GSM) hot path.  TEST INFRASTRUCTURE ONLY.

This module is the plain, slow, obviously-correct statement of what the CUDA path must compute.  It is
imported only by ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference``
legs of ``bench.py``.  It shares no code with ``paper_1501_01752_b200/`` and never imports it.

Everything is complex fp64 (paper: "double precision").  No FFT is used anywhere here:
the Toeplitz product is the O(n^2) sum written out, the voxel harmonics are a direct DFT, tiny systems
are assembled densely and solved by LU (numpy.linalg.solve), larger ones by a textbook full GMRES.

Conventions:
  * orders m_a in {-M..M}, M=(N-1)/2 for odd N; {-N/2..N/2-1} for even N              (R1)
  * E(r) = sum_m E_m exp(+i k_m.r), eps(r) = sum_d eps_d exp(+i G_d.r)                 (R3)
  * units eps0 = mu0 = c = 1: k_b^2 = k0^2 eps_b, k0 = omega/c                        (R4)
  * plain Laurent rule, no inverse-rule reformulation                                  (R6)
  * field layout x[c, i1, i2, i3], i_a = m_a - m_a,min
  * coefficient layout c[d1+N1-1, d2+N2-1, d3+N3-1], |d_a| <= N_a-1

Pins (tests/test_oracle_*.py): sphere closed form vs direct DFT of a voxelised sphere; homogeneous cell;
uniform-cell closed form; Rytov laminate dispersion + arithmetic/harmonic-mean limits; dense brute force;
Green-dyadic eigen-identities; Hermitian-pencil eigenproblem at the pole; synthetic pole recovery;
Maxwell-Garnett values and printed n_eff of the paper (tests/golden/).  No function here is unpinned.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

SPHERE, ELLIPSOID, BOX, POLYHEDRON = 0, 1, 2, 3


# --------------------------------------------------------------------------------------------------
# orders and lattice
# --------------------------------------------------------------------------------------------------
def order_range(N: int) -> np.ndarray:
    """Harmonic indices kept along one axis (reading R1)."""
    if N % 2 == 1:
        M = (N - 1) // 2
        return np.arange(-M, M + 1)
    return np.arange(-N // 2, N // 2)


def reciprocal_periods(periods) -> np.ndarray:
    """K_a = 2 pi / Lambda_a."""
    return 2.0 * np.pi / np.asarray(periods, dtype=np.float64)


# --------------------------------------------------------------------------------------------------
# a0: permittivity harmonics (Delta eps / eps_b)_d
# --------------------------------------------------------------------------------------------------
def _sphere_form(x: np.ndarray) -> np.ndarray:
    """3 (sin x - x cos x) / x^3, -> 1 at x = 0 (Fourier image of the unit ball, textbook)."""
    out = np.ones_like(x)
    big = np.abs(x) > 1e-4
    xb = x[big]
    out[big] = 3.0 * (np.sin(xb) - xb * np.cos(xb)) / xb**3
    xs = x[~big]
    out[~big] = 1.0 - xs**2 / 10.0 + xs**4 / 280.0
    return out


def _sinc(t: np.ndarray) -> np.ndarray:
    """sin t / t, -> 1 at 0."""
    out = np.ones_like(t)
    nz = np.abs(t) > 1e-300
    out[nz] = np.sin(t[nz]) / t[nz]
    return out


def polyhedron_image(G, vertices, faces) -> complex:
    """int_P exp(-i G.r) d^3r for a polyhedron with planar faces ("Fourier images of sphere and
    polyhedron"; the paper prints no formula - this is the divergence theorem applied twice, textbook):

        G != 0:  (i / |G|^2) sum_faces (G.n_f) I_f,            I_f = int_face exp(-i G.r) dS
        I_f   =  (i / |G_t|^2) sum_edges (G_t.m_e) L_e exp(-i G.c_e) sinc(G.(b - a) / 2)      if G_t != 0
              =  A_f exp(-i G.r_f)                                                            if G_t = 0
    with n_f the outward unit normal, G_t = G - (G.n_f) n_f, and for every edge a -> b of the face (vertices listed
    counter-clockwise seen from outside): length L_e, midpoint c_e, in-plane outward normal m_e = t_e x n_f.
    G = 0 gives the volume, (1/3) sum_faces (r_f.n_f) A_f."""
    G = np.asarray(G, dtype=np.float64)
    V = np.asarray(vertices, dtype=np.float64)
    g2 = float(G @ G)
    total = 0.0 + 0.0j
    for f in faces:
        P = V[list(f)]
        nvec = np.zeros(3)
        for k in range(1, len(P) - 1):                           # area vector of the fan triangulation
            nvec += 0.5 * np.cross(P[k] - P[0], P[k + 1] - P[0])
        area = float(np.linalg.norm(nvec))
        n = nvec / area
        if g2 == 0.0:
            total += float(P[0] @ n) * area / 3.0
            continue
        Gn = float(G @ n)
        Gt = G - Gn * n
        gt2 = float(Gt @ Gt)
        if gt2 < 1e-18 * g2:
            If = area * np.exp(-1j * float(G @ P[0]))
        else:
            If = 0.0 + 0.0j
            for k in range(len(P)):
                a, b = P[k], P[(k + 1) % len(P)]
                L = float(np.linalg.norm(b - a))
                m = np.cross((b - a) / L, n)
                If += float(Gt @ m) * L * np.exp(-1j * float(G @ (a + b)) / 2) * np.sinc(float(G @ (b - a)) / 2 / np.pi)
            If *= 1j / gt2
        total += 1j / g2 * Gn * If
    return complex(total)


def coeffs_analytic(periods, orders, shapes, eps_bg=1.0, eps_b=None) -> np.ndarray:
    """c_d = (1/V) int_cell (eps(r)-eps_b)/eps_b exp(-i G_d.r) d^3r for superposed analytic shapes.

    shapes: list of dicts {kind, center(3), size(3), eps}.  size = (R, -, -) for a sphere, semi-axes for
    an ellipsoid, full widths for a box; a polyhedron carries `vertices` (relative to the centre) and `faces`
    (vertex index lists, counter-clockwise seen from outside) instead.  c_d = delta_d0 (eps_bg-eps_b)/eps_b
        + sum_i (eps_i-eps_bg)/eps_b * f_i * S_i(d) * exp(-i G_d.r_c,i).
    """
    eps_b = eps_bg if eps_b is None else eps_b
    periods = np.asarray(periods, dtype=np.float64)
    K = reciprocal_periods(periods)
    N1, N2, N3 = orders
    d1 = np.arange(-(N1 - 1), N1)[:, None, None] * K[0]
    d2 = np.arange(-(N2 - 1), N2)[None, :, None] * K[1]
    d3 = np.arange(-(N3 - 1), N3)[None, None, :] * K[2]
    G1, G2, G3 = np.broadcast_arrays(d1, d2, d3)
    vol = float(np.prod(periods))
    c = np.zeros(G1.shape, dtype=np.complex128)
    c[N1 - 1, N2 - 1, N3 - 1] = (eps_bg - eps_b) / eps_b
    for s in shapes:
        kind, ctr, size, eps_i = s["kind"], np.asarray(s["center"], float), np.asarray(s["size"], float), s["eps"]
        delta = (eps_i - eps_bg) / eps_b
        if kind == SPHERE:
            f = 4.0 / 3.0 * np.pi * size[0] ** 3 / vol
            S = _sphere_form(np.sqrt(G1**2 + G2**2 + G3**2) * size[0])
        elif kind == ELLIPSOID:
            f = 4.0 / 3.0 * np.pi * size[0] * size[1] * size[2] / vol
            S = _sphere_form(np.sqrt((G1 * size[0]) ** 2 + (G2 * size[1]) ** 2 + (G3 * size[2]) ** 2))
        elif kind == BOX:
            f = float(np.prod(size)) / vol
            S = _sinc(G1 * size[0] / 2) * _sinc(G2 * size[1] / 2) * _sinc(G3 * size[2] / 2)
        elif kind == POLYHEDRON:                                 # vertices relative to the centre; f S = image / V_cell
            f = 1.0 / vol
            S = np.empty(G1.shape, dtype=np.complex128)
            for idx in np.ndindex(G1.shape):
                S[idx] = polyhedron_image((G1[idx], G2[idx], G3[idx]), s["vertices"], s["faces"])
        else:
            raise ValueError("unknown shape kind")
        phase = np.exp(-1j * (G1 * ctr[0] + G2 * ctr[1] + G3 * ctr[2]))
        c += delta * f * S * phase
    return c


def coeffs_voxel(eps_grid: np.ndarray, orders, eps_b=1.0) -> np.ndarray:
    """Direct DFT of a voxel grid: c_d = (1/Nv^3) sum_j (eps_j-eps_b)/eps_b exp(-2 pi i sum_a d_a j_a/Nv_a).

    Written as three successive axis sums with explicit exp matrices (still a direct DFT, no FFT);
    tests cross-check it against `coeffs_voxel_single` (the literal triple sum).  Requires Nv_a >= 2N_a-1.
    """
    g = (np.asarray(eps_grid, dtype=np.complex128) - eps_b) / eps_b
    out = g
    for ax, (N, Nv) in enumerate(zip(orders, g.shape)):
        if Nv < 2 * N - 1:
            raise ValueError("voxel grid too coarse for the requested orders")
        d = np.arange(-(N - 1), N)
        W = np.exp(-2j * np.pi * np.outer(d, np.arange(Nv)) / Nv) / Nv        # [2N-1, Nv]
        out = np.moveaxis(np.tensordot(W, out, axes=([1], [ax])), 0, ax)
    return out


def coeffs_voxel_single(eps_grid: np.ndarray, d, eps_b=1.0) -> complex:
    """One coefficient by the literal triple sum (tiny grids only)."""
    g = (np.asarray(eps_grid, dtype=np.complex128) - eps_b) / eps_b
    Nv = g.shape
    acc = 0.0 + 0.0j
    for j1 in range(Nv[0]):
        for j2 in range(Nv[1]):
            for j3 in range(Nv[2]):
                ph = d[0] * j1 / Nv[0] + d[1] * j2 / Nv[1] + d[2] * j3 / Nv[2]
                acc += g[j1, j2, j3] * np.exp(-2j * np.pi * ph)
    return acc / (Nv[0] * Nv[1] * Nv[2])


# --------------------------------------------------------------------------------------------------
# a1-a4: Toeplitz product (T x)_{c,m} = sum_m' c_{m-m'} x_{c,m'}                      PAPER.md:50, Eq. 4
# --------------------------------------------------------------------------------------------------
def toeplitz_row(c: np.ndarray, x: np.ndarray, i) -> np.ndarray:
    """All three components of (T x) at one output harmonic i=(i1,i2,i3): the sum over m' written out.

    c_{m-m'} with m-m' = i-i' sits at c[i1-i1'+N1-1, ...]; over i1' = 0..N1-1 that is the slice
    c[i1+N1-1 : i1-1 : -1] (reversed window).
    """
    N1, N2, N3 = x.shape[1:]
    i1, i2, i3 = i
    w = c[i1 : i1 + N1, i2 : i2 + N2, i3 : i3 + N3][::-1, ::-1, ::-1]       # w[i'] = c[i - i' + N - 1]
    return np.tensordot(x, w, axes=([1, 2, 3], [0, 1, 2]))


def toeplitz_matvec(c: np.ndarray, x: np.ndarray) -> np.ndarray:
    """(T x) for every harmonic, O(n^2), no FFT and no stored matrix."""
    N1, N2, N3 = x.shape[1:]
    y = np.empty_like(x)
    for i1 in range(N1):
        for i2 in range(N2):
            for i3 in range(N3):
                y[:, i1, i2, i3] = toeplitz_row(c, x, (i1, i2, i3))
    return y


_clib = None


def _load_clib():
    """oracle/toeplitz_oracle.c compiled by __graft_entry__.build() (plain C triple loop + OpenMP)."""
    global _clib
    if _clib is None:
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libtoeplitz_oracle.so")
        if not os.path.exists(path):
            raise RuntimeError("oracle C helper not built: run python -c 'import __graft_entry__ as g; g.build_oracle()'")
        lib = ctypes.CDLL(path)
        lib.toeplitz_matvec_c.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p] + [ctypes.c_int] * 3
        lib.toeplitz_matvec_c.restype = None
        lib.oracle_num_threads.restype = ctypes.c_int
        _clib = lib
    return _clib


def toeplitz_matvec_c(c: np.ndarray, x: np.ndarray) -> np.ndarray:
    """Same O(n^2) sum in plain C (used where the numpy loop is too slow; pinned to `toeplitz_matvec`)."""
    lib = _load_clib()
    c = np.ascontiguousarray(c, dtype=np.complex128)
    x = np.ascontiguousarray(x, dtype=np.complex128)
    y = np.empty_like(x)
    N1, N2, N3 = x.shape[1:]
    lib.toeplitz_matvec_c(c.ctypes.data, x.ctypes.data, y.ctypes.data, N1, N2, N3)
    return y


def num_threads() -> int:
    return int(_load_clib().oracle_num_threads())


# --------------------------------------------------------------------------------------------------
# a5: Green dyadic and the operator A x = x - G (T x)
# --------------------------------------------------------------------------------------------------
def wavevectors(periods, orders, k_inc) -> np.ndarray:
    """k_m = k_inc + (m1 K1, m2 K2, m3 K3), shape [3, N1, N2, N3]."""
    K = reciprocal_periods(periods)
    m1, m2, m3 = (order_range(N) for N in orders)
    k = np.empty((3,) + tuple(orders), dtype=np.float64)
    k[0] = (k_inc[0] + m1 * K[0])[:, None, None]
    k[1] = (k_inc[1] + m2 * K[1])[None, :, None]
    k[2] = (k_inc[2] + m3 * K[2])[None, None, :]
    return k


def green_multiply(F: np.ndarray, periods, k_inc, k0, eps_b) -> np.ndarray:
    """(G F)_{a,m} = sum_b (k_b^2 delta_ab - k_am k_bm)/(k_m.k_m - k_b^2) F_{b,m}   (Eq. 4)."""
    k = wavevectors(periods, F.shape[1:], k_inc)
    kb2 = k0 * k0 * eps_b
    s = k[0] * F[0] + k[1] * F[1] + k[2] * F[2]
    den = k[0] ** 2 + k[1] ** 2 + k[2] ** 2 - kb2
    return (kb2 * F - k * s[None]) / den[None]


def apply_operator(c, x, periods, k_inc, k0, eps_b, matvec=toeplitz_matvec) -> np.ndarray:
    """y = x - G (T x): the left-hand side of Eq. 4 moved to one side."""
    return x - green_multiply(matvec(c, x), periods, k_inc, k0, eps_b)


def incident(orders, pol) -> np.ndarray:
    """b_{c,m} = a_c delta_{m,0}."""
    b = np.zeros((3,) + tuple(orders), dtype=np.complex128)
    i0 = tuple(int(np.where(order_range(N) == 0)[0][0]) for N in orders)
    b[(slice(None),) + i0] = np.asarray(pol, dtype=np.complex128)
    return b


def zero_order(E: np.ndarray) -> np.ndarray:
    """xi: the three components of E at m = 0."""
    i0 = tuple(int(np.where(order_range(N) == 0)[0][0]) for N in E.shape[1:])
    return E[(slice(None),) + i0].copy()


# --------------------------------------------------------------------------------------------------
# dense assembly + LU (tiny n)                                                        brute force
# --------------------------------------------------------------------------------------------------
def assemble_dense(c, periods, orders, k_inc, k0, eps_b) -> np.ndarray:
    """A = I - G T as a dense (3n x 3n) matrix, row/col index = ((c*N1+i1)*N2+i2)*N3+i3."""
    N1, N2, N3 = orders
    n = N1 * N2 * N3
    i1, i2, i3 = np.meshgrid(np.arange(N1), np.arange(N2), np.arange(N3), indexing="ij")
    i1, i2, i3 = i1.ravel(), i2.ravel(), i3.ravel()
    T = c[(i1[:, None] - i1[None, :]) + N1 - 1, (i2[:, None] - i2[None, :]) + N2 - 1, (i3[:, None] - i3[None, :]) + N3 - 1]
    k = wavevectors(periods, orders, k_inc).reshape(3, n)
    kb2 = k0 * k0 * eps_b
    den = (k**2).sum(axis=0) - kb2
    A = np.eye(3 * n, dtype=np.complex128)
    for a in range(3):
        for b in range(3):
            g = ((kb2 if a == b else 0.0) - k[a] * k[b]) / den                  # G_{m;ab}
            A[a * n : (a + 1) * n, b * n : (b + 1) * n] -= g[:, None] * T
    return A


def solve_dense(c, periods, orders, k_inc, k0, eps_b, pol) -> np.ndarray:
    A = assemble_dense(c, periods, orders, k_inc, k0, eps_b)
    b = incident(orders, pol).ravel()
    return np.linalg.solve(A, b).reshape((3,) + tuple(orders))


# --------------------------------------------------------------------------------------------------
# a6-a8: full GMRES, modified Gram-Schmidt, Givens least squares       PAPER.md:105 (Saad [27], Alg. 6.9)
# --------------------------------------------------------------------------------------------------
def gmres(apply, b: np.ndarray, tol: float, max_iters: int, x0: np.ndarray | None = None):
    """Unrestarted GMRES (reading R9).  <u,v> = sum conj(u) v.

    x0 = None: start from zero.  x0 given (the solution at the neighbouring kappa point of the
    equidistant mesh): textbook form - r0 = b - A x0, GMRES on A d = r0, x = x0 + d (Saad Alg. 6.9
    with a non-zero initial guess).  The stop test stays relative to ||b||, so every start meets the same bar.

    Returns (x, history, iters): history[j] = |g_{j+1}| / ||b|| after iteration j+1.
    Lucky breakdown (h_{j+1,j} <= eps ||A v_j||: nothing of A v_j is left after orthogonalisation) exits as converged
    (reading R23; the test is scale-free, so it acts the same for a guessed start with a tiny ||r0||).
    """
    shape = b.shape
    bv = b.ravel()
    bnorm = np.linalg.norm(bv)
    if bnorm == 0.0:
        return np.zeros(shape, np.complex128), [], 0
    if x0 is None:
        xs = np.zeros_like(bv)
        r0 = bv
    else:
        xs = np.asarray(x0, dtype=np.complex128).ravel().copy()
        r0 = bv - apply(xs.reshape(shape)).ravel()
    beta = np.linalg.norm(r0)
    if beta <= tol * bnorm:
        return xs.reshape(shape), [], 0
    V = [r0 / beta]
    H = np.zeros((max_iters + 1, max_iters), dtype=np.complex128)
    cs = np.zeros(max_iters)
    sn = np.zeros(max_iters, dtype=np.complex128)
    g = np.zeros(max_iters + 1, dtype=np.complex128)
    g[0] = beta
    hist = []
    m = 0
    for j in range(max_iters):
        w = apply(V[j].reshape(shape)).ravel().copy()
        for i in range(j + 1):                                   # modified Gram-Schmidt
            H[i, j] = np.vdot(V[i], w)
            w -= H[i, j] * V[i]
        hn = np.linalg.norm(w)
        H[j + 1, j] = hn
        wnorm = np.linalg.norm(H[: j + 2, j])                    # ||A v_j|| (Pythagoras over v_0..v_j and the remainder)
        for i in range(j):                                       # previous rotations on the new column
            t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
            H[i + 1, j] = -np.conj(sn[i]) * H[i, j] + cs[i] * H[i + 1, j]
            H[i, j] = t
        a, bb = H[j, j], H[j + 1, j]
        r = np.sqrt(abs(a) ** 2 + abs(bb) ** 2)
        if r == 0.0:
            cs[j], sn[j] = 1.0, 0.0
        elif abs(a) == 0.0:
            cs[j], sn[j] = 0.0, 1.0
        else:
            cs[j] = abs(a) / r
            sn[j] = (a / abs(a)) * np.conj(bb) / r
        H[j, j] = cs[j] * a + sn[j] * bb
        H[j + 1, j] = 0.0
        g[j + 1] = -np.conj(sn[j]) * g[j]
        g[j] = cs[j] * g[j]
        m = j + 1
        hist.append(abs(g[j + 1]) / bnorm)
        if hist[-1] <= tol or hn <= np.finfo(float).eps * wnorm:
            break
        V.append(w / hn)
    y = np.zeros(m, dtype=np.complex128)
    for i in range(m - 1, -1, -1):                               # back substitution
        y[i] = (g[i] - H[i, i + 1 : m] @ y[i + 1 : m]) / H[i, i]
    x = xs.copy()
    for i in range(m):
        x += y[i] * V[i]
    return x.reshape(shape), hist, m


def solve_gmres(c, periods, orders, k_inc, k0, eps_b, pol, tol=1e-13, max_iters=200, matvec=None, x0=None):
    """Solve Eq. 4 by full GMRES with the O(n^2) Toeplitz product.  Returns (E, history, iters)."""
    mv = matvec or toeplitz_matvec
    b = incident(orders, pol)
    return gmres(lambda v: apply_operator(c, v, periods, k_inc, k0, eps_b, mv), b, tol, max_iters, x0)


# --------------------------------------------------------------------------------------------------
# a10: pole search and retrieval                                      PAPER.md:64-95 (Eq. 6-10), R11-R16
# --------------------------------------------------------------------------------------------------
def pole_search(kappa, xi, Np=5, Nd=10):
    """Poles eta_j and amplitudes zeta_j of xi(kappa) ~ sum zeta_j/(kappa-eta_j) + regular part.

    Eq. 8/9 with xi in the NUMERATOR (reading R11): for each sliding window of Nd+1 points the Nd-th divided
    difference of P(kappa) xi(kappa) vanishes; sum_k [sum_i t_i^k xi_i w_i] p_k = - sum_i t_i^Np xi_i w_i,
    w_i = 1/prod_{j!=i}(t_i - t_j).  All windows (>= Np of them, R13) are used, least squares if more.
    kappa is mapped affinely to t in [-1, 1] before forming powers (R16).  Roots = eigenvalues of the
    companion matrix.  Amplitudes by Eq. 10 over the window nearest to each pole (R12).
    """
    kappa = np.asarray(kappa, dtype=np.float64)
    xi = np.asarray(xi, dtype=np.complex128)
    npts = len(kappa)
    S = npts - Nd
    if S < Np:
        raise ValueError("need at least Np + Nd points")
    mid, half = 0.5 * (kappa[0] + kappa[-1]), 0.5 * (kappa[-1] - kappa[0])
    t = (kappa - mid) / half
    M = np.zeros((S, Np), dtype=np.complex128)
    rhs = np.zeros(S, dtype=np.complex128)
    for s in range(S):
        tw, xw = t[s : s + Nd + 1], xi[s : s + Nd + 1]
        w = np.array([1.0 / np.prod(np.delete(tw[i] - tw, i)) for i in range(Nd + 1)])
        for k in range(Np):
            M[s, k] = np.sum(tw**k * xw * w)
        rhs[s] = -np.sum(tw**Np * xw * w)
    scale = np.abs(M).max()
    # Eq. 9 is a plain linear system for p_k; solve it in the least-squares sense by QR WITHOUT rank
    # truncation.  A rank-revealing pseudo-inverse (numpy.linalg.lstsq) returns the minimum-norm solution when the
    # window sees fewer than Np poles, which makes all Np roots coalesce at the pole and amplifies rounding as
    # eps^(1/Np); the untruncated solution keeps the true pole as a simple root and lets the spurious ones wander.
    Q, R = np.linalg.qr(M / scale)
    p = np.linalg.solve(R, Q.conj().T @ (rhs / scale))
    comp = np.zeros((Np, Np), dtype=np.complex128)               # companion of t^Np + sum p_k t^k
    comp[1:, :-1] = np.eye(Np - 1)
    comp[:, -1] = -p
    eta_t = np.linalg.eigvals(comp)
    zeta_t = np.zeros(Np, dtype=np.complex128)
    for k in range(Np):
        s = int(np.clip(np.argmin(np.abs(t - eta_t[k].real)) - Nd // 2, 0, S - 1))
        tw, xw = t[s : s + Nd + 1], xi[s : s + Nd + 1]
        acc = 0.0 + 0.0j
        for i in range(Nd + 1):
            P_i = np.prod(tw[i] - eta_t)
            lag = np.prod(np.delete(eta_t[k] - tw, i) / np.delete(tw[i] - tw, i))
            acc += xw[i] * P_i * lag
        zeta_t[k] = acc / np.prod(np.delete(eta_t[k] - eta_t, k))
    return mid + half * eta_t, half * zeta_t


def select_pole(eta, zeta, lo, hi):
    """Root with Re eta in [lo, hi] and the largest |zeta| (reading R15).  Returns its index or -1."""
    best, amp = -1, -1.0
    for j in range(len(eta)):
        if lo <= eta[j].real <= hi and abs(zeta[j]) > amp:
            best, amp = j, abs(zeta[j])
    return best


def retrieve_eps(eta, k0):
    """n_eff = eta / k0, eps_eff = n_eff^2."""
    n = eta / k0
    return n, n * n


# --------------------------------------------------------------------------------------------------
# H-field formulation, Eq. 5                         SURVEY 8(f) "next" item 1
# --------------------------------------------------------------------------------------------------
# H_m = H^inc_m + k_m x [ sum_m' D_{m-m'} (k_m' x H_m') ] / (k_b^2 - k_m.k_m),  D_d = delta_d0 - (eps_b/eps)_d.
# (The Levi-Civita sums of Eq. 5 are the two cross products.)  The coefficients of the INVERSE permittivity are
# "found analytically just in the same way": for inclusions eps_i in a background eps_bg,
#   1 - eps_b/eps(r) = (1 - eps_b/eps_bg) + sum_i (eps_b/eps_bg - eps_b/eps_i) chi_i(r)
# (exact for non-overlapping inclusions; overlapping ones superpose their terms, as in coeffs_analytic).
def coeffs_inverse_analytic(periods, orders, shapes, eps_bg=1.0, eps_b=None) -> np.ndarray:
    """D_d = Fourier coefficients of 1 - eps_b/eps(r), same layout as coeffs_analytic."""
    eps_b = eps_bg if eps_b is None else eps_b
    unit = [dict(s, eps=1.0) for s in shapes]
    N1, N2, N3 = orders
    D = np.zeros((2 * N1 - 1, 2 * N2 - 1, 2 * N3 - 1), dtype=np.complex128)
    D[N1 - 1, N2 - 1, N3 - 1] = 1.0 - eps_b / eps_bg
    for s, s1 in zip(shapes, unit):
        # f S(d) exp(-i G.r_c) of this shape alone = coeffs_analytic with unit contrast (eps = 1, bg = 0, eps_b = 1)
        form = coeffs_analytic(periods, orders, [s1], eps_bg=0.0, eps_b=1.0)
        form[N1 - 1, N2 - 1, N3 - 1] += 1.0      # remove that call's background term (0 - 1)/1 at d = 0
        D += (eps_b / eps_bg - eps_b / s["eps"]) * form
    return D


def coeffs_inverse_voxel(eps_grid: np.ndarray, orders, eps_b=1.0) -> np.ndarray:
    """Direct DFT of 1 - eps_b/eps_j (same three axis sums as coeffs_voxel)."""
    g = 1.0 - eps_b / np.asarray(eps_grid, dtype=np.complex128)
    # coeffs_voxel forms (grid - eps_b)/eps_b; feed it a grid whose image under that map is g
    return coeffs_voxel(eps_b * (g + 1.0), orders, eps_b)


def cross_k(k: np.ndarray, F: np.ndarray) -> np.ndarray:
    """(k_m x F_m) for every harmonic; k real [3, N1, N2, N3], F complex [3, N1, N2, N3]."""
    return np.stack([k[1] * F[2] - k[2] * F[1], k[2] * F[0] - k[0] * F[2], k[0] * F[1] - k[1] * F[0]])


def apply_operator_H(D, x, periods, k_inc, k0, eps_b, matvec=toeplitz_matvec) -> np.ndarray:
    """y = x - k x T_D(k x x) / (k_b^2 - k.k): Eq. 5 with the unknown moved to one side."""
    k = wavevectors(periods, x.shape[1:], k_inc)
    kb2 = k0 * k0 * eps_b
    den = kb2 - (k[0] ** 2 + k[1] ** 2 + k[2] ** 2)
    return x - cross_k(k, matvec(D, cross_k(k, x))) / den[None]


def assemble_dense_H(D, periods, orders, k_inc, k0, eps_b) -> np.ndarray:
    """Dense matrix of Eq. 5, same index convention as assemble_dense, built entry by entry from the Levi-Civita form:
    A[(a,m),(v,m')] = delta - sum_{b,g,s} xi_abg k_bm / (k_b^2 - k_m^2) D_{m-m'} xi_gsv k_sm'."""
    N1, N2, N3 = orders
    n = N1 * N2 * N3
    i1, i2, i3 = np.meshgrid(np.arange(N1), np.arange(N2), np.arange(N3), indexing="ij")
    i1, i2, i3 = i1.ravel(), i2.ravel(), i3.ravel()
    T = D[(i1[:, None] - i1[None, :]) + N1 - 1, (i2[:, None] - i2[None, :]) + N2 - 1, (i3[:, None] - i3[None, :]) + N3 - 1]
    k = wavevectors(periods, orders, k_inc).reshape(3, n)
    den = k0 * k0 * eps_b - (k**2).sum(axis=0)
    xi = np.zeros((3, 3, 3))
    xi[0, 1, 2] = xi[1, 2, 0] = xi[2, 0, 1] = 1.0
    xi[0, 2, 1] = xi[2, 1, 0] = xi[1, 0, 2] = -1.0
    A = np.eye(3 * n, dtype=np.complex128)
    for a in range(3):
        for v in range(3):
            blk = np.zeros((n, n), dtype=np.complex128)
            for b in range(3):
                for g_ in range(3):
                    if xi[a, b, g_] == 0.0:
                        continue
                    for s in range(3):
                        if xi[g_, s, v] == 0.0:
                            continue
                        blk += xi[a, b, g_] * xi[g_, s, v] * (k[b] / den)[:, None] * T * k[s][None, :]
            A[a * n : (a + 1) * n, v * n : (v + 1) * n] -= blk
    return A


def solve_dense_H(D, periods, orders, k_inc, k0, eps_b, pol) -> np.ndarray:
    A = assemble_dense_H(D, periods, orders, k_inc, k0, eps_b)
    return np.linalg.solve(A, incident(orders, pol).ravel()).reshape((3,) + tuple(orders))


def solve_gmres_H(D, periods, orders, k_inc, k0, eps_b, pol, tol=1e-13, max_iters=200, matvec=None):
    mv = matvec or toeplitz_matvec
    return gmres(lambda v: apply_operator_H(D, v, periods, k_inc, k0, eps_b, mv), incident(orders, pol), tol, max_iters)


def retrieve_two_stage(xi_of_kappa, k0, n_lo, n_hi, ncoarse=29, nfine=18, fine_step=0.002, Np=5, Nd=10):
    """Two-stage retrieval of one effective index (reading R16).

    xi_of_kappa(kappa_array) -> complex responses.  Stage 1: equidistant coarse mesh on [n_lo, n_hi] k0, pole search,
    estimate eta_c.  Stage 2: nfine (even) points spaced fine_step k0, centred so that eta_c falls mid-way between the
    two middle nodes, pole search.  Returns (n_eff, eps_eff, zeta)."""
    coarse = np.linspace(n_lo, n_hi, ncoarse) * k0
    eta, zeta = pole_search(coarse, xi_of_kappa(coarse), Np, Nd)
    b = select_pole(eta, zeta, coarse[0], coarse[-1])
    if b < 0:
        raise RuntimeError("no pole inside the coarse window")
    fine = eta[b].real + fine_step * k0 * (np.arange(nfine) - 0.5 * (nfine - 1))
    eta, zeta = pole_search(fine, xi_of_kappa(fine), Np, Nd)
    b = select_pole(eta, zeta, fine[0], fine[-1])
    if b < 0:
        raise RuntimeError("no pole inside the fine window")
    n, eps = retrieve_eps(eta[b], k0)
    return n, eps, zeta[b]
