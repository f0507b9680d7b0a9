"""Writes tests/golden/config1_closed_form.txt: for BASELINE.json config 1 (64x64 uniform periodic grid,
n = 1, gamma = 1/2, 10 scales) the energies e_l = 1/2 <phibar_l^2> of the CLOSED-FORM filtered field

    phibar_l = sum_j a_j cos(2 pi m_j.x/N + theta_j) / (1 + gamma l^2 lambda_mj),
    lambda_m = 4 - 2 cos(2 pi m_x/N) - 2 cos(2 pi m_y/N)        (h = 1)

(eq. (1), applied to eigenvectors of the 5-point Laplacian).  Uses only the input
generator (workloads/); nothing from the oracle's solver and nothing from the CUDA path.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from workloads import make_config  # noqa: E402

w = make_config(1)
N = 64
wv = w.waves[0]
lam = 4.0 - 2.0 * np.cos(2 * np.pi * wv.k[:, 0] / N) - 2.0 * np.cos(2 * np.pi * wv.k[:, 1] / N)
basis = np.cos(w.mesh.coords @ (wv.k.T * wv.scale) + wv.theta)
rows = []
for ell in w.ells:
    ref = basis @ (wv.amp / (1.0 + 0.5 * ell ** 2 * lam))
    rows.append((ell, 0.5 * np.mean(ref ** 2)))
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_closed_form.txt")
np.savetxt(out, np.array(rows), fmt="%.17e",
           header="config 1 closed-form energies (PAPER.md:33 eq.(1) on plane waves; PAPER.md:75): ell  e_ell")
print("wrote", out)
