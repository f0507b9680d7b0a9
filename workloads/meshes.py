"""Seeded synthetic triangular meshes (inputs only: no filter arithmetic lives here).

Stand-ins for the meshes of the paper, which are not available offline: the regular grid split
into two triangles per cell (Fig. 2), the synthetic Cartesian and
spherical timing meshes (Fig. 6) and the >10 M-vertex FESOM2 surface mesh
(PAPER.md:133).  The recipes are those of SURVEY.md section 8(d) and readings
A12-A13; DESIGN.md restates them.

Every generator returns a `Mesh` holding plain numpy arrays:
  coords  float64 [V][dim]   vertex positions (dim = 2 planar, 3 sphere)
  tri     int32   [T][3]     vertex ids of each triangle
  period  float64 [dim] or None   period per axis (0 = not periodic)
  h       float              nominal edge length ("one edge length" of BASELINE.json configs)
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np


@dataclass
class Mesh:
    coords: np.ndarray
    tri: np.ndarray
    period: Optional[np.ndarray]
    h: float
    name: str = ""

    @property
    def n_vert(self) -> int:
        return int(self.coords.shape[0])

    @property
    def n_tri(self) -> int:
        return int(self.tri.shape[0])

    @property
    def dim(self) -> int:
        return int(self.coords.shape[1])


# --------------------------------------------------------------------------- planar grids
def grid_mesh(n: int, *, periodic: bool = True, jitter: float = 0.0, random_diagonals: bool = False,
              rng: Optional[np.random.Generator] = None, h: float = 1.0) -> Mesh:
    """n x n cells, each split into two triangles (Fig. 2).

    periodic=True : n*n vertices, vertex id = iy*n + ix at (ix*h, iy*h), period (n*h, n*h).
    periodic=False: (n+1)*(n+1) vertices, id = iy*(n+1) + ix.
    jitter        : each vertex displaced by U(-jitter, jitter)*h in x and in y.
    random_diagonals: per cell the diagonal is v00-v11 or v10-v01 with probability 1/2;
                      otherwise always v00-v11 (config 1: "along the same diagonal").
    """
    if rng is None:
        rng = np.random.default_rng(0)
    nv1 = n if periodic else n + 1
    iy, ix = np.meshgrid(np.arange(nv1), np.arange(nv1), indexing="ij")
    coords = np.stack([ix.ravel(), iy.ravel()], axis=1).astype(np.float64) * h
    # draw order is fixed: jitter first, then diagonals
    if jitter > 0.0:
        coords = coords + rng.uniform(-jitter, jitter, size=coords.shape) * h
    cy, cx = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    cx = cx.ravel()
    cy = cy.ravel()
    if periodic:
        x1 = (cx + 1) % n
        y1 = (cy + 1) % n
    else:
        x1 = cx + 1
        y1 = cy + 1
    v00 = cy * nv1 + cx
    v10 = cy * nv1 + x1
    v01 = y1 * nv1 + cx
    v11 = y1 * nv1 + x1
    if random_diagonals:
        flip = rng.integers(0, 2, size=cx.shape[0]).astype(bool)
    else:
        flip = np.zeros(cx.shape[0], dtype=bool)
    # diagonal v00-v11: (v00,v10,v11),(v00,v11,v01);  diagonal v10-v01: (v00,v10,v01),(v10,v11,v01)
    ta = np.where(flip[:, None], np.stack([v00, v10, v01], 1), np.stack([v00, v10, v11], 1))
    tb = np.where(flip[:, None], np.stack([v10, v11, v01], 1), np.stack([v00, v11, v01], 1))
    tri = np.empty((2 * cx.shape[0], 3), dtype=np.int32)
    tri[0::2] = ta
    tri[1::2] = tb
    period = np.array([n * h, n * h], dtype=np.float64) if periodic else None
    return Mesh(coords=np.ascontiguousarray(coords), tri=tri, period=period, h=h,
                name=f"grid{n}{'p' if periodic else ''}")


def equilateral_mesh(nx: int, ny: int, h: float = 1.0) -> Mesh:
    """Periodic lattice of equilateral triangles (ny even).  Used only as a textbook special case:
    every off-diagonal stiffness entry is -1/sqrt(3) and every dual area sqrt(3)/2 h^2."""
    assert ny % 2 == 0
    iy, ix = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    x = (ix + 0.5 * (iy % 2)) * h
    y = iy * (np.sqrt(3.0) / 2.0) * h
    coords = np.stack([x.ravel(), y.ravel()], 1)

    def vid(jx, jy):
        return (jy % ny) * nx + (jx % nx)

    tris = []
    for jy in range(ny):
        for jx in range(nx):
            if jy % 2 == 0:
                a, b, c, d = vid(jx, jy), vid(jx + 1, jy), vid(jx, jy + 1), vid(jx - 1, jy + 1)
                tris.append((a, b, c))
                tris.append((a, c, d))
            else:
                a, b, c, d = vid(jx, jy), vid(jx + 1, jy), vid(jx + 1, jy + 1), vid(jx, jy + 1)
                tris.append((a, b, c))
                tris.append((a, c, d))
    period = np.array([nx * h, ny * (np.sqrt(3.0) / 2.0) * h])
    return Mesh(coords=coords, tri=np.asarray(tris, dtype=np.int32), period=period, h=h,
                name=f"equi{nx}x{ny}")


# --------------------------------------------------------------------------- icosphere
def _icosahedron():
    t = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
                  [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
                  [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    return v, f


def icosphere_edge(level: int) -> float:
    """Nominal edge h_L: edge of the equilateral triangle whose area is the mean flat triangle area
    4*pi/(20*4^L) of the unit sphere (SURVEY.md reading A10)."""
    return float(np.sqrt(16.0 * np.pi / (np.sqrt(3.0) * 20.0 * 4.0 ** level)))


def icosphere(level: int) -> Mesh:
    """Unit icosphere by `level` midpoint subdivisions with re-projection.
    V = 10*4^L + 2, T = 20*4^L.  Vertex numbering is the construction order (12 base vertices, then
    the edge midpoints of each level): an arbitrary, locality-poor numbering like a model's."""
    v, f = _icosahedron()
    for _ in range(level):
        nv = v.shape[0]
        a = np.concatenate([f[:, 0], f[:, 1], f[:, 2]])
        b = np.concatenate([f[:, 1], f[:, 2], f[:, 0]])
        lo = np.minimum(a, b)
        hi = np.maximum(a, b)
        key = lo * np.int64(nv) + hi
        uniq, inv = np.unique(key, return_inverse=True)
        ulo = uniq // nv
        uhi = uniq - ulo * nv
        mid = v[ulo] + v[uhi]
        mid /= np.linalg.norm(mid, axis=1, keepdims=True)
        v = np.concatenate([v, mid], axis=0)
        nt = f.shape[0]
        m01 = nv + inv[0:nt]
        m12 = nv + inv[nt:2 * nt]
        m20 = nv + inv[2 * nt:3 * nt]
        f = np.concatenate([np.stack([f[:, 0], m01, m20], 1),
                            np.stack([f[:, 1], m12, m01], 1),
                            np.stack([f[:, 2], m20, m12], 1),
                            np.stack([m01, m12, m20], 1)], axis=0)
    return Mesh(coords=np.ascontiguousarray(v), tri=f.astype(np.int32), period=None,
                h=icosphere_edge(level), name=f"icosphere{level}")


def jitter_sphere(mesh: Mesh, amount: float, rng: np.random.Generator) -> Mesh:
    """Displace every vertex tangentially by U(-amount, amount)^2 * h in a local tangent basis and
    re-project onto the unit sphere (BASELINE.json configs 3-5)."""
    x = mesh.coords
    # helper axis: the coordinate axis least aligned with x
    k = np.argmin(np.abs(x), axis=1)
    a = np.zeros_like(x)
    a[np.arange(x.shape[0]), k] = 1.0
    e1 = np.cross(x, a)
    e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
    e2 = np.cross(x, e1)
    u = rng.uniform(-amount, amount, size=(x.shape[0], 2)) * mesh.h
    y = x + u[:, 0:1] * e1 + u[:, 1:2] * e2
    y /= np.linalg.norm(y, axis=1, keepdims=True)
    return Mesh(coords=np.ascontiguousarray(y), tri=mesh.tri, period=None, h=mesh.h,
                name=mesh.name + "j")


def land_mask(mesh: Mesh, positions: np.ndarray, fraction: float, rng: np.random.Generator,
              n_modes: int = 32) -> Mesh:
    """Remove `fraction` of the vertices as random smooth blobs (SURVEY.md reading A13):
    g(x) = sum_j cos(kappa_j . x + theta_j), kappa_j isotropic, |kappa_j| ~ U(2, 8), evaluated at
    `positions` (the unjittered vertices); vertices with g below its `fraction` quantile are removed,
    every triangle touching a removed vertex is dropped (the remaining boundary edges then carry the
    natural no-flux condition), vertices left in no triangle are dropped, and ids are
    compacted in increasing order."""
    d = rng.normal(size=(n_modes, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    kappa = d * rng.uniform(2.0, 8.0, size=(n_modes, 1))
    theta = rng.uniform(0.0, 2.0 * np.pi, size=n_modes)
    g = np.zeros(positions.shape[0])
    step = 1 << 18
    for s in range(0, positions.shape[0], step):
        g[s:s + step] = np.cos(positions[s:s + step] @ kappa.T + theta).sum(axis=1)
    n_remove = int(round(fraction * positions.shape[0]))
    order = np.argsort(g, kind="stable")
    keep_v = np.ones(positions.shape[0], dtype=bool)
    keep_v[order[:n_remove]] = False
    tri = mesh.tri
    keep_t = keep_v[tri[:, 0]] & keep_v[tri[:, 1]] & keep_v[tri[:, 2]]
    tri = tri[keep_t]
    used = np.zeros(positions.shape[0], dtype=bool)
    used[tri.ravel()] = True
    new_id = np.cumsum(used, dtype=np.int64) - 1
    tri = new_id[tri].astype(np.int32)
    return Mesh(coords=np.ascontiguousarray(mesh.coords[used]), tri=np.ascontiguousarray(tri),
                period=None, h=mesh.h, name=mesh.name + "m")


# --------------------------------------------------------------------------- unstructured planar (Delaunay)
def delaunay_mesh(n: int, rng: np.random.Generator, hubs: int = 3, hub_valence: int = 14) -> Mesh:
    """Non-periodic planar mesh of the square [0, n]^2 with unit point density: a regular boundary (spacing 1),
    uniformly random interior points and `hubs` hub vertices, each the centre of a circle of `hub_valence` points
    with nothing else inside (so the hub has exactly that many neighbours), triangulated by scipy's Delaunay.
    Vertex valences spread from 3 to hub_valence -- unlike the grids and icospheres, whose rows never exceed 8
    entries -- which is what a general unstructured mesh looks like to the SELL packing."""
    from scipy.spatial import Delaunay
    t = np.arange(n, dtype=np.float64)
    border = np.concatenate([np.stack([t, np.zeros(n)], 1), np.stack([np.full(n, float(n)), t], 1),
                             np.stack([n - t, np.full(n, float(n))], 1), np.stack([np.zeros(n), n - t], 1)])
    inner = rng.uniform(0.7, n - 0.7, size=((n - 1) * (n - 1), 2))
    centres = rng.uniform(0.25 * n, 0.75 * n, size=(hubs, 2))
    rad = 1.5
    for c in centres:
        inner = inner[np.linalg.norm(inner - c, axis=1) > rad + 0.35]
    ang = 2.0 * np.pi * np.arange(hub_valence) / hub_valence
    rings = [c + rad * np.stack([np.cos(ang + 0.1 * i), np.sin(ang + 0.1 * i)], 1) for i, c in enumerate(centres)]
    pts = np.concatenate([border, inner, centres] + rings)
    tri = Delaunay(pts).simplices.astype(np.int32)
    return Mesh(coords=np.ascontiguousarray(pts), tri=np.ascontiguousarray(tri), period=None, h=1.0,
                name=f"delaunay{n}")


def sphere_band(mesh: Mesh, max_lat_deg: float) -> Mesh:
    """Keep the part of a sphere mesh with |latitude| <= max_lat_deg: every triangle touching a removed vertex is
    dropped, ids are compacted.  Model meshes keep their grid poles out of the ocean (a rotated grid with
    the pole over land); the lon/lat components of a velocity, which the vector filter of PAPER.md:87-91 works
    with, are singular at the poles (metric factor m = tan(latitude) / R_e)."""
    x = mesh.coords
    lat = np.degrees(np.arcsin(x[:, 2] / np.linalg.norm(x, axis=1)))
    keep_v = np.abs(lat) <= max_lat_deg
    tri = mesh.tri
    tri = tri[keep_v[tri[:, 0]] & keep_v[tri[:, 1]] & keep_v[tri[:, 2]]]
    used = np.zeros(x.shape[0], dtype=bool)
    used[tri.ravel()] = True
    new_id = np.cumsum(used, dtype=np.int64) - 1
    return Mesh(coords=np.ascontiguousarray(x[used]), tri=np.ascontiguousarray(new_id[tri].astype(np.int32)),
                period=None, h=mesh.h, name=mesh.name + f"b{max_lat_deg:g}")
