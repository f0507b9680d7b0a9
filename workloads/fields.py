"""Seeded synthetic scalar fields and scale lists (inputs only: no filter arithmetic lives here).

Stand-ins for the FESOM2 velocity components of PAPER.md:133 (not available offline): sums of random
plane waves with amplitude |k|^-1.5 (BASELINE.json configs; SURVEY.md reading A14).  Each generator also
returns the wave parameters so a test can evaluate closed forms for them.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class Waves:
    k: np.ndarray        # [J][dim] integer wavevectors (lattice units for planar, rad/unit for sphere)
    amp: np.ndarray      # [J]
    theta: np.ndarray    # [J]
    scale: float         # phase = scale * (k . x) + theta


def _eval_waves(coords: np.ndarray, w: Waves) -> np.ndarray:
    """phi(x) = sum_j amp_j cos(scale * k_j.x + theta_j), chunked over vertices."""
    out = np.empty(coords.shape[0], dtype=np.float64)
    kt = np.ascontiguousarray(w.k.T.astype(np.float64)) * w.scale
    try:
        import torch
        ktt = torch.from_numpy(kt)
        th = torch.from_numpy(w.theta)
        am = torch.from_numpy(w.amp)
        xs = torch.from_numpy(np.ascontiguousarray(coords))
        o = torch.from_numpy(out)
        step = 1 << 16
        for s in range(0, coords.shape[0], step):
            ph = xs[s:s + step] @ ktt
            ph += th
            torch.cos_(ph)
            o[s:s + step] = ph @ am
    except ImportError:  # pragma: no cover - numpy path gives the same numbers to rounding
        step = 1 << 15
        for s in range(0, coords.shape[0], step):
            out[s:s + step] = np.cos(coords[s:s + step] @ kt + w.theta) @ w.amp
    return out


def planar_wave_field(coords: np.ndarray, n: int, kmax: int, n_waves: int,
                      rng: np.random.Generator, h: float = 1.0):
    """phi(x) = sum_j |m_j|^-1.5 cos(2 pi m_j.x/(n h) + theta_j); m_j drawn without replacement,
    uniformly from the integer lattice points with 1 <= |m| <= kmax; theta_j ~ U[0, 2 pi)."""
    r = np.arange(-kmax, kmax + 1)
    mx, my = np.meshgrid(r, r, indexing="ij")
    m2 = mx * mx + my * my
    sel = (m2 >= 1) & (m2 <= kmax * kmax)
    cand = np.stack([mx[sel], my[sel]], 1)
    pick = rng.choice(cand.shape[0], size=n_waves, replace=False)
    k = cand[pick].astype(np.int64)
    theta = rng.uniform(0.0, 2.0 * np.pi, size=n_waves)
    amp = np.sqrt((k * k).sum(1).astype(np.float64)) ** -1.5
    w = Waves(k=k, amp=amp, theta=theta, scale=2.0 * np.pi / (n * h))
    return _eval_waves(coords, w), w


def sphere_wave_field(coords: np.ndarray, kmax: int, n_waves: int, rng: np.random.Generator):
    """phi(x) = sum_j |kappa_j|^-1.5 cos(kappa_j.x + theta_j); kappa_j integer 3-vectors uniform in
    1 <= |kappa| <= kmax (rejection from the cube, duplicates allowed); theta_j ~ U[0, 2 pi)."""
    ks = []
    need = n_waves
    while need > 0:
        c = rng.integers(-kmax, kmax + 1, size=(4 * need + 16, 3))
        n2 = (c * c).sum(1)
        c = c[(n2 >= 1) & (n2 <= kmax * kmax)]
        ks.append(c[:need])
        need -= ks[-1].shape[0]
    k = np.concatenate(ks, 0).astype(np.int64)
    theta = rng.uniform(0.0, 2.0 * np.pi, size=n_waves)
    amp = np.sqrt((k * k).sum(1).astype(np.float64)) ** -1.5
    w = Waves(k=k, amp=amp, theta=theta, scale=1.0)
    return _eval_waves(coords, w), w


def log_spaced(lo: float, hi: float, count: int) -> np.ndarray:
    """l_j = lo (hi/lo)^(j/(count-1)), both ends included (SURVEY.md reading A15)."""
    if count == 1:
        return np.array([lo], dtype=np.float64)
    j = np.arange(count, dtype=np.float64)
    return lo * (hi / lo) ** (j / (count - 1))


def sphere_frames(coords: np.ndarray):
    """Unit zonal (east) and meridional (north) vectors at points of a sphere centred at the origin."""
    x = coords / np.linalg.norm(coords, axis=1, keepdims=True)
    rho = np.sqrt(x[:, 0] ** 2 + x[:, 1] ** 2)
    east = np.stack([-x[:, 1] / rho, x[:, 0] / rho, np.zeros_like(rho)], 1)
    north = np.cross(x, east)
    return east, north


def sphere_velocity_field(coords: np.ndarray, kmax: int, n_waves: int, rng: np.random.Generator):
    """Seeded tangent velocity field on the sphere in zonal / meridional components (u, v): the tangential part of
    U(x) = sum_j |kappa_j|^-1.5 cos(kappa_j.x + theta_j) b_j with random unit vectors b_j, plus a rigid rotation about
    a random axis (amplitude 1).  Stand-in for the FESOM2 surface velocities of PAPER.md:133."""
    k = rng.integers(-kmax, kmax + 1, size=(4 * n_waves + 16, 3))
    n2 = (k * k).sum(1)
    k = k[(n2 >= 1) & (n2 <= kmax * kmax)][:n_waves].astype(np.float64)
    theta = rng.uniform(0.0, 2.0 * np.pi, size=k.shape[0])
    b = rng.normal(size=(k.shape[0], 3))
    b /= np.linalg.norm(b, axis=1, keepdims=True)
    amp = np.sqrt((k * k).sum(1)) ** -1.5
    axis = rng.normal(size=3)
    axis /= np.linalg.norm(axis)
    U = np.cross(axis[None, :], coords)
    step = 1 << 15
    for s in range(0, coords.shape[0], step):
        U[s:s + step] += (np.cos(coords[s:s + step] @ k.T + theta) * amp) @ b
    east, north = sphere_frames(coords)
    return np.einsum("ij,ij->i", U, east), np.einsum("ij,ij->i", U, north)
