"""The seeded input generators (workloads/): reproducible bit for bit, whatever the number of threads (DESIGN.md
section 3), and what they promise about the fields (closed form of the plane-wave sum)."""
import os
import subprocess
import sys
import hashlib

import numpy as np

from workloads import fields as wf
from workloads import make_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _digest(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def test_wave_sum_does_not_depend_on_the_number_of_threads(monkeypatch):
    rng = np.random.default_rng(5)
    coords = rng.uniform(0.0, 300.0, size=(3 * wf._EVAL_STEP + 777, 2))      # several chunks and a ragged tail
    w = wf.Waves(k=rng.integers(-40, 41, size=(96, 2)), amp=rng.uniform(0.1, 1.0, 96),
                 theta=rng.uniform(0.0, 6.28, 96), scale=2.0 * np.pi / 300.0)
    many = wf._eval_waves(coords, w)
    monkeypatch.setattr(os, "sched_getaffinity", lambda pid: {0}, raising=False)      # one thread: the serial loop
    one = wf._eval_waves(coords, w)
    assert np.array_equal(many, one)
    # the definition, element by element, on a sample (pairwise vs plain summation: rounding only)
    for v in (0, 1, wf._EVAL_STEP - 1, wf._EVAL_STEP, coords.shape[0] - 1):
        want = sum(w.amp[j] * np.cos(w.scale * float(w.k[j] @ coords[v]) + w.theta[j]) for j in range(96))
        assert abs(many[v] - want) <= 1e-12 * np.abs(w.amp).sum()


def test_config_fields_are_the_same_in_a_fresh_process():
    here = make_config(1)
    code = ("import sys, hashlib; sys.path.insert(0, %r); from workloads import make_config; w = make_config(1); "
            "print(hashlib.sha256(w.fields.tobytes()).hexdigest(), hashlib.sha256(w.mesh.coords.tobytes()).hexdigest())" % ROOT)
    env = dict(os.environ, OMP_NUM_THREADS="3")        # a different thread setting must not matter either
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, check=True).stdout.split()
    assert out == [_digest(here.fields), _digest(here.mesh.coords)]
    # zero mean: a sum of lattice plane waves over the full periodic grid cancels exactly up to rounding
    assert abs(here.fields.sum()) <= 1e-11 * np.abs(here.fields).sum()


def test_velocity_field_is_reproducible():
    from workloads import icosphere, sphere_band, sphere_velocity_field
    mesh = sphere_band(icosphere(3), 70.0)          # lon/lat components are singular at the poles
    u1, v1 = sphere_velocity_field(mesh.coords, 12, 40, np.random.default_rng(3))
    u2, v2 = sphere_velocity_field(mesh.coords, 12, 40, np.random.default_rng(3))
    assert np.array_equal(u1, u2) and np.array_equal(v1, v2)
    assert np.isfinite(u1).all() and np.isfinite(v1).all() and np.abs(u1).max() > 0.1
