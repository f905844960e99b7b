"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module holds NO arithmetic of the method: only geometry descriptions, scan lists and seeded random
vectors.  It serves both the CUDA path and the CPU oracle (tests feed the same objects to each side) and
imports neither.  Length unit: the vacuum wavelength lambda = 1, so k0 = 2 pi unless stated.

Stand-ins: the paper measures on lattices of spheres / cubes whose exact radius,
period and wavevector are not all printed; BASELINE.json's five configs fix them, and these generators
reproduce those configs.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SPHERE, ELLIPSOID, BOX, POLYHEDRON = 0, 1, 2, 3
TWO_PI = 2.0 * math.pi
SEED = 150101752


@dataclass
class Geometry:
    """One periodic cell: periods, Fourier orders and either analytic shapes or a voxel grid."""
    name: str
    periods: tuple
    orders: tuple
    shapes: list = field(default_factory=list)     # dicts {kind, center, size, eps}
    eps_bg: complex = 1.0
    eps_b: complex = 1.0
    voxels: np.ndarray | None = None               # complex128 [Nv1, Nv2, Nv3], i3 fastest
    fft_grid: tuple = ()                           # unused placeholder (the FFT grid is the library's choice: Plan.info())

    @property
    def n(self) -> int:
        return int(np.prod(self.orders))


def _geo(name, periods, orders, shapes=None, eps_bg=1.0, eps_b=1.0, voxels=None) -> Geometry:
    return Geometry(name, tuple(periods), tuple(orders), shapes or [], eps_bg, eps_b, voxels, ())


def sphere_lattice(orders=(7, 7, 7), period=0.2, radius_frac=0.3, eps=4.0, eps_bg=1.0) -> Geometry:
    """Config 1 (W1): simple cubic lattice, one sphere per cell, radius 0.3 Lambda, Lambda = 0.2 lambda."""
    L = period
    return _geo("sphere", (L, L, L), orders,
                [dict(kind=SPHERE, center=(0, 0, 0), size=(radius_frac * L, 0, 0), eps=eps)], eps_bg, eps_bg)


def laminate(orders=(1, 1, 63), fill=0.5, eps_slab=9.0, eps_bg=1.0) -> Geometry:
    """Config 2 (W2): slabs eps=1 / eps=9 stacked along z; length unit = Lambda_z (so k0 = 2 pi Lambda_z/lambda)."""
    return _geo("laminate", (1.0, 1.0, 1.0), orders,
                [dict(kind=BOX, center=(0, 0, 0), size=(1.0, 1.0, fill), eps=eps_slab)], eps_bg, eps_bg)


def ellipsoid_lattice(orders=(15, 15, 15)) -> Geometry:
    """Config 3 (W3): orthorhombic cell (0.2, 0.25, 0.3) lambda, ellipsoid semi-axes (0.35,0.25,0.15).Lambda_a (R18)."""
    per = (0.2, 0.25, 0.3)
    semi = (0.35 * per[0], 0.25 * per[1], 0.15 * per[2])
    return _geo("ellipsoid", per, orders, [dict(kind=ELLIPSOID, center=(0, 0, 0), size=semi, eps=12.0)])


def woodpile(orders=(31, 31, 31), period=0.3, eps_rod=6.25) -> Geometry:
    """Config 4 (W4): four layers of rectangular rods, w = h = Lambda/4, alternating x/y, half-period offset (R19)."""
    L, w = period, period / 4
    shapes = [
        dict(kind=BOX, center=(0.0, 0.0, 1 * L / 8), size=(L, w, w), eps=eps_rod),       # x-rod
        dict(kind=BOX, center=(0.0, 0.0, 3 * L / 8), size=(w, L, w), eps=eps_rod),       # y-rod
        dict(kind=BOX, center=(0.0, L / 2, 5 * L / 8), size=(L, w, w), eps=eps_rod),     # x-rod, shifted
        dict(kind=BOX, center=(L / 2, 0.0, 7 * L / 8), size=(w, L, w), eps=eps_rod),     # y-rod, shifted
    ]
    return _geo("woodpile", (L, L, L), orders, shapes)


def polyhedron(name: str, scale: float = 1.0, rotate=None):
    """Vertices and faces (counter-clockwise seen from outside) of a few convex and one non-convex test polyhedron.
    rotate = (axis[3], angle): rigid rotation, so that faces are not aligned with the lattice."""
    if name == "tetrahedron":
        v = np.array([(1, 1, 1), (1, -1, -1), (-1, 1, -1), (-1, -1, 1)], dtype=float)
        faces = [(0, 1, 2), (0, 3, 1), (0, 2, 3), (1, 3, 2)]
    elif name == "cube":
        v = np.array([(x, y, z) for x in (-1, 1) for y in (-1, 1) for z in (-1, 1)], dtype=float)
        faces = [(0, 1, 3, 2), (4, 6, 7, 5), (0, 4, 5, 1), (2, 3, 7, 6), (0, 2, 6, 4), (1, 5, 7, 3)]
    elif name == "octahedron":
        v = np.array([(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)], dtype=float)
        faces = [(0, 2, 4), (2, 1, 4), (1, 3, 4), (3, 0, 4), (2, 0, 5), (1, 2, 5), (3, 1, 5), (0, 3, 5)]
    elif name == "lshape":          # non-convex prism: L-shaped cross-section extruded along z
        xy = [(-1, -1), (1, -1), (1, 0), (0, 0), (0, 1), (-1, 1)]
        v = np.array([(x, y, z) for z in (-0.5, 0.5) for (x, y) in xy], dtype=float)
        faces = [tuple(range(5, -1, -1)), tuple(range(6, 12))] + [(k, (k + 1) % 6, 6 + (k + 1) % 6, 6 + k) for k in range(6)]
    else:
        raise ValueError(name)
    v = v * scale
    if rotate is not None:
        ax, ang = np.asarray(rotate[0], dtype=float), float(rotate[1])
        ax = ax / np.linalg.norm(ax)
        Kx = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
        R = np.eye(3) + math.sin(ang) * Kx + (1 - math.cos(ang)) * (Kx @ Kx)
        v = v @ R.T
    return v, [tuple(int(i) for i in f) for f in faces]


def polyhedron_lattice(orders=(7, 7, 7), name="octahedron", period=0.2, scale=0.07, eps=6.0, center=(0.0, 0.0, 0.0),
                       rotate=((1.0, 2.0, 3.0), 0.4)) -> Geometry:
    """Cubic lattice of one dielectric polyhedron per cell (analytic Fourier image of a polyhedron)."""
    v, faces = polyhedron(name, scale, rotate)
    return _geo(f"poly-{name}", (period,) * 3, orders,
                [dict(kind=POLYHEDRON, center=center, size=(0, 0, 0), eps=eps, vertices=v, faces=faces)])


def random_spheres(seed=SEED, count=20, period=0.25):
    """The 20 (centre, radius, eps) triples of config 5, drawn once from a seeded generator (R20)."""
    rng = np.random.default_rng(seed)
    centers = rng.uniform(0.0, period, size=(count, 3))
    radii = rng.uniform(0.05, 0.15, size=count) * period
    eps = rng.uniform(2.0, 10.0, size=count)
    return centers, radii, eps


def voxel_composite(orders=(31, 31, 31), nv=128, seed=SEED, period=0.25) -> Geometry:
    """Config 5 (W5): union of 20 seeded spheres voxelised on nv^3 (later spheres overwrite, minimum image)."""
    centers, radii, eps = random_spheres(seed, 20, period)
    ax = np.arange(nv) * (period / nv)
    grid = np.ones((nv, nv, nv), dtype=np.complex128)
    for ctr, R, e in zip(centers, radii, eps):
        d = [np.abs(ax - ctr[a]) for a in range(3)]
        d = [np.minimum(t, period - t) for t in d]
        r2 = d[0][:, None, None] ** 2 + d[1][None, :, None] ** 2 + d[2][None, None, :] ** 2
        grid[r2 <= R * R] = e
    return _geo("voxel", (period,) * 3, orders, voxels=grid)


def cavity_lattice(orders, kind, n_host, period=0.3) -> Geometry:
    """PAPER.md:135/:139 worked examples: air cube (side Lambda/2) or sphere (R = 0.125 lambda) cavities."""
    L = period
    if kind == "cube":
        shape = dict(kind=BOX, center=(0, 0, 0), size=(L / 2, L / 2, L / 2), eps=1.0)
    else:
        shape = dict(kind=SPHERE, center=(0, 0, 0), size=(0.125, 0, 0), eps=1.0)
    e = n_host * n_host
    return _geo(f"{kind}-cavity", (L, L, L), orders, [shape], e, e)


def tetragonal_cavities(ratio, orders=(7, 7, 7), radius=0.02, fill=4.0 / 3.0 * math.pi / 27.0, n_host=1.5) -> Geometry:
    """PAPER.md:127, :143 (Fig. 4): spherical air cavities of radius `radius` (in wavelengths) in a host of index 1.5 on a
    simple tetragonal lattice, Lambda_x = ratio * Lambda_y,z, at the constant filling factor f = (4/3) pi / 27 = 0.155
    (R = Lambda / 3 at equal periods): Lambda_y,z = (4 pi R^3 / (3 f ratio))^(1/3).  ratio = 1 is the isotropic crystal."""
    lt = (4.0 / 3.0 * math.pi * radius ** 3 / (fill * ratio)) ** (1.0 / 3.0)
    e = n_host * n_host
    return _geo(f"tetragonal-{ratio:g}", (ratio * lt, lt, lt), orders,
                [dict(kind=SPHERE, center=(0, 0, 0), size=(radius, 0, 0), eps=1.0)], e, e)


def normal_surface_lines(count, seed=SEED):
    """Cross-section of the Fresnel normal surface by the xz plane: `count` seeded propagation
    directions s = (sin t, 0, cos t), each with the two transverse unit amplitudes - y (normal to the plane: the ordinary
    sheet of a crystal whose axis is x) and y x s (in the plane: the extraordinary sheet).  Returns (dirs [2 count, 3],
    pols [2 count, 3]), the two sheets of direction i at rows 2 i and 2 i + 1."""
    rng = np.random.default_rng(seed + 5)
    t = np.sort(rng.uniform(0.1, 0.5 * math.pi - 0.1, count))
    dirs, pols = [], []
    for ti in t:
        s = np.array([math.sin(ti), 0.0, math.cos(ti)])
        dirs += [s, s]
        pols += [np.array([0.0, 1.0, 0.0]), np.cross([0.0, 1.0, 0.0], s)]
    return np.array(dirs), np.array(pols)


# ---- scan lists -----------------------------------------------------------------------------------
DIRECTIONS = {
    # tensor entry <- (propagation axis, polarisation axis): reading R14 (cyclic)
    "xx": (2, 0),
    "yy": (0, 1),
    "zz": (1, 2),
}


def kappa_mesh(n_lo, n_hi, npts, k0=TWO_PI) -> np.ndarray:
    """Equidistant mesh of |k_inc| = n_i k0."""
    return np.linspace(n_lo, n_hi, npts) * k0


def scan_points(kappa, prop_axis, pol_axis, k0=TWO_PI):
    """(k_bloch[npts,3], k0[npts], pol[npts,6]) for a kappa mesh along one axis with one polarisation."""
    kappa = np.asarray(kappa, dtype=np.float64)
    kb = np.zeros((len(kappa), 3))
    kb[:, prop_axis] = kappa
    pol = np.zeros((len(kappa), 6))
    pol[:, 2 * pol_axis] = 1.0
    return kb, np.full(len(kappa), float(k0)), pol


def direction_sweep(count, seed=SEED):
    """Direction sweep at fixed omega: `count` seeded unit vectors s and, for each,
    the transverse unit amplitude a = s x z / |s x z|.  Returns a list of (s[3], a[3])."""
    rng = np.random.default_rng(seed + 4)
    out = []
    for _ in range(count):
        v = rng.standard_normal(3)
        s = v / np.linalg.norm(v)
        a = np.cross(s, [0.0, 0.0, 1.0])
        out.append((s, a / np.linalg.norm(a)))
    return out


def random_field(batch, orders, seed=SEED) -> np.ndarray:
    """Seeded complex standard-normal x[batch, 3, N1, N2, N3] for operator-apply tests."""
    rng = np.random.default_rng(seed)
    shape = (batch, 3) + tuple(orders)
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex128)
