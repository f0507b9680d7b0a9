"""Seeded synthetic scalar fields and scale lists (inputs only: no filter arithmetic lives here).

Stand-ins for the FESOM2 velocity components of PAPER.md:133 (not available offline): sums of random
plane waves with amplitude |k|^-1.5 (BASELINE.json configs; SURVEY.md reading A14).  Each generator also
returns the wave parameters so a test can evaluate closed forms for them.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np


@dataclass
class Waves:
    k: np.ndarray        # [J][dim] integer wavevectors (lattice units for planar, rad/unit for sphere)
    amp: np.ndarray      # [J]
    theta: np.ndarray    # [J]
    scale: float         # phase = scale * (k . x) + theta


def _cos_phases(x, kt, theta):
    """cos(x . k_j + theta_j) for a chunk of points x [m][dim] and wavevectors kt [dim][J]: elementwise operations only."""
    ph = np.multiply.outer(x[:, 0], kt[0])
    for d in range(1, x.shape[1]):
        ph += np.multiply.outer(x[:, d], kt[d])
    ph += theta
    np.cos(ph, out=ph)
    return ph


def _eval_chunk(coords, kt, theta, amp, out, s, e):
    c = _cos_phases(coords[s:e], kt, theta)
    c *= amp
    out[s:e] = c.sum(axis=1)


_EVAL_STEP = 2048        # vertices per chunk: fixed, so that the arithmetic does not depend on the number of threads


def _eval_waves(coords: np.ndarray, w: Waves) -> np.ndarray:
    """phi(x) = sum_j amp_j cos(scale * k_j.x + theta_j).

    Bit-reproducible from run to run: every value is a fixed sequence of elementwise numpy operations (products and sums
    of the phase in coordinate order, cos, the weighted sum over the waves in numpy's fixed pairwise order) on chunks of
    a fixed size; threads only share out the chunks.  No BLAS and no multithreaded library kernel is involved: an
    earlier form (torch CPU matmul / cos_) gave fields that differed by 1e-10 in a few percent of processes on a
    16-thread host, which showed as changed iteration counts on the finite-termination case of config 1."""
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    out = np.empty(coords.shape[0], dtype=np.float64)
    kt = np.ascontiguousarray(w.k.T.astype(np.float64)) * w.scale
    theta = np.ascontiguousarray(w.theta, dtype=np.float64)
    amp = np.ascontiguousarray(w.amp, dtype=np.float64)
    starts = range(0, coords.shape[0], _EVAL_STEP)
    try:
        n_threads = len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        n_threads = os.cpu_count() or 1
    n_threads = max(1, min(n_threads, 32, len(starts)))

    def run(s):
        _eval_chunk(coords, kt, theta, amp, out, s, min(s + _EVAL_STEP, coords.shape[0]))

    if n_threads == 1:
        for s in starts:
            run(s)
    else:
        with ThreadPoolExecutor(n_threads) as pool:
            list(pool.map(run, starts))
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
    kt = np.ascontiguousarray(k.T)
    for s in range(0, coords.shape[0], _EVAL_STEP):        # same fixed-order elementwise evaluation as _eval_waves
        c = _cos_phases(coords[s:s + _EVAL_STEP], kt, theta)
        c *= amp
        for d in range(3):
            U[s:s + _EVAL_STEP, d] += (c * b[:, d]).sum(axis=1)
    east, north = sphere_frames(coords)
    return np.einsum("ij,ij->i", U, east), np.einsum("ij,ij->i", U, north)
