"""The five BASELINE.json configurations as seeded synthetic inputs (inputs only).

Seeds follow SURVEY.md section 8(d): SeedSequence(20240407*10 + config) spawned into the streams
`mesh`, `mask`, `field_0`, `field_1`, ... in that order.  `make_config(i)` builds config i (1-based, as
BASELINE.json lists them); the keyword overrides build geometrically similar smaller cases for tests
that the CPU oracle can finish in seconds (the wavenumber cut-off is scaled with the mesh).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

from . import fields as F
from . import meshes as M

BASE_SEED = 20240407 * 10


@dataclass
class Workload:
    config: int
    mesh: M.Mesh
    fields: np.ndarray          # [F][V] float64
    ells: np.ndarray            # [L] float64, absolute lengths (coordinate units), ascending
    order_n: int                # filter order n (1 harmonic, 2 biharmonic)
    waves: List[F.Waves] = field(default_factory=list)
    note: str = ""

    @property
    def n_rhs(self) -> int:
        return int(self.fields.shape[0] * self.ells.shape[0])


def _streams(config: int, n_fields: int, offset: int = 0):
    ss = np.random.SeedSequence(BASE_SEED + config)
    kids = ss.spawn(2 + offset + n_fields)
    kids = kids[:2] + kids[2 + offset:]
    return [np.random.default_rng(k) for k in kids]


def make_config(config: int, *, n: Optional[int] = None, level: Optional[int] = None,
                n_fields: Optional[int] = None, n_ells: Optional[int] = None,
                ell_max: Optional[float] = None, field_offset: int = 0) -> Workload:
    """`field_offset` skips that many field streams: fields [offset, offset + n_fields) of the same seeded sequence
    (what rank r of a multi-GPU run generates for itself)."""
    if config == 1:
        n = 64 if n is None else n
        nf = 1 if n_fields is None else n_fields
        rs = _streams(1, nf, field_offset)
        mesh = M.grid_mesh(n, periodic=True, rng=rs[0])
        fl, wv = zip(*[F.planar_wave_field(mesh.coords, n, n // 2, min(128, 2 * n), rs[2 + i])
                       for i in range(nf)])
        ells = F.log_spaced(1.0, float(n // 2) if ell_max is None else ell_max,
                            10 if n_ells is None else n_ells)
        return Workload(1, mesh, np.stack(fl), ells, 1, list(wv), "uniform periodic grid")
    if config == 2:
        n = 512 if n is None else n
        nf = 2 if n_fields is None else n_fields
        rs = _streams(2, nf, field_offset)
        mesh = M.grid_mesh(n, periodic=True, jitter=0.3, random_diagonals=True, rng=rs[0])
        fl, wv = zip(*[F.planar_wave_field(mesh.coords, n, n // 2, 128, rs[2 + i]) for i in range(nf)])
        ells = F.log_spaced(1.0, float(n // 2) if ell_max is None else ell_max,
                            20 if n_ells is None else n_ells)
        return Workload(2, mesh, np.stack(fl), ells, 1, list(wv), "jittered periodic grid, random diagonals")
    if config == 3:
        level = 9 if level is None else level
        nf = 1 if n_fields is None else n_fields
        rs = _streams(3, nf, field_offset)
        mesh = M.jitter_sphere(M.icosphere(level), 0.25, rs[0])
        kmax = max(4, int(round(400 * 2.0 ** (level - 9))))
        fl, wv = zip(*[F.sphere_wave_field(mesh.coords, kmax, 512, rs[2 + i]) for i in range(nf)])
        # n = 2: scales 1-32 edge lengths (SURVEY.md reading A16)
        ells = mesh.h * F.log_spaced(1.0, 32.0 if ell_max is None else ell_max,
                                     20 if n_ells is None else n_ells)
        return Workload(3, mesh, np.stack(fl), ells, 2, list(wv), "jittered icosphere, biharmonic")
    if config in (4, 5):
        level = 10 if level is None else level
        nf = (2 if config == 4 else 8) if n_fields is None else n_fields
        # configs 4 and 5 share one mesh ("same 10.5M-vertex masked sphere"): mesh and mask streams of config 4
        rs_mesh = _streams(4, 0)
        base = M.icosphere(level)
        jit = M.jitter_sphere(base, 0.25, rs_mesh[0])
        mesh = M.land_mask(jit, base.coords, 0.30, rs_mesh[1])
        rs = _streams(config, nf, field_offset)
        kmax = max(4, int(round(800 * 2.0 ** (level - 10))))
        fl, wv = zip(*[F.sphere_wave_field(mesh.coords, kmax, 512, rs[2 + i]) for i in range(nf)])
        if config == 4:
            lmax = min(1000.0, 1000.0 * 2.0 ** (level - 10)) if ell_max is None else ell_max
            ells = mesh.h * F.log_spaced(1.0, max(lmax, 2.0), 40 if n_ells is None else n_ells)
            return Workload(4, mesh, np.stack(fl), ells, 1, list(wv), "masked jittered icosphere, harmonic")
        ells = mesh.h * F.log_spaced(1.0, 32.0 if ell_max is None else ell_max,
                                     40 if n_ells is None else n_ells)
        return Workload(5, mesh, np.stack(fl), ells, 2, list(wv), "masked jittered icosphere, biharmonic")
    raise ValueError(f"config must be 1..5, got {config}")
