"""Pins of the oracle's vector filter with metric terms against things other than itself (CPU only).

  * the integrals of PAPER.md:89-91 evaluated in the test by quadrature with explicit P1 basis functions (affine
    functions from an inverted vertex matrix, edge-midpoint rule, exact for quadratics) -- not the oracle's closed forms;
  * T antisymmetric, D~ symmetric, D_2 = [D~ T; -T D~] symmetric positive semidefinite;
  * a planar mesh has no metric terms: the vector filter is two scalar filters;
  * dense direct solve (numpy) of the 2V x 2V system built in the test;
  * rigid rotations are eigenfields of the vector (Hodge) Laplacian on the sphere with eigenvalue 2 / R^2, as the l = 1
    harmonics are for the scalar one: attenuation 1 / (1 + gamma (2 l^2 / R^2)^n) -- about the z axis (u only) and about
    an axis in the equatorial plane (u and v, coupled through T: a wrong sign of T fails here).
"""
import numpy as np
import pytest

from workloads import grid_mesh, icosphere, jitter_sphere, sphere_band, sphere_frames, sphere_velocity_field

GAMMA = 0.5


def metric_matrices_by_quadrature(coords, tri, radius):
    """Dense D~ / l^2, T / l^2 and the lumped mass from the definitions: per flat triangle an orthonormal in-plane frame,
    N_i affine with N_i(x_j) = delta_ij, integrals by the edge-midpoint rule; m = tan(lat) / R and the zonal direction
    at the centroid."""
    nv = coords.shape[0]
    D = np.zeros((nv, nv))
    T = np.zeros((nv, nv))
    A = np.zeros(nv)
    for t in tri:
        X = coords[t]
        e1 = X[1] - X[0]
        e1 = e1 / np.linalg.norm(e1)
        w = X[2] - X[0]
        w = w - np.dot(w, e1) * e1
        e2 = w / np.linalg.norm(w)
        q = np.array([[np.dot(p - X[0], e1), np.dot(p - X[0], e2)] for p in X])
        B = np.linalg.inv(np.column_stack([np.ones(3), q]))          # column i: (a, gx, gy) of N_i
        area = 0.5 * abs(q[1, 0] * q[2, 1] - q[1, 1] * q[2, 0])
        cen = X.mean(axis=0)
        if coords.shape[1] == 3 and radius > 0:
            lat = np.arcsin(cen[2] / np.linalg.norm(cen))
            m = np.tan(lat) / radius
            east3 = np.array([-cen[1], cen[0], 0.0]) / np.hypot(cen[0], cen[1])
            east = np.array([np.dot(east3, e1), np.dot(east3, e2)])    # in-plane components
            curv = 1.0 / radius ** 2
        else:
            m, east, curv = 0.0, np.array([1.0, 0.0]), 0.0
        mids = [0.5 * (q[0] + q[1]), 0.5 * (q[1] + q[2]), 0.5 * (q[2] + q[0])]
        N = lambda i, p: B[0, i] + B[1, i] * p[0] + B[2, i] * p[1]
        for i in range(3):
            gi = B[1:, i]
            A[t[i]] += sum(N(i, p) for p in mids) * area / 3.0          # int N_i = lumped mass share
            for j in range(3):
                gj = B[1:, j]
                nn = sum(N(i, p) * N(j, p) for p in mids) * area / 3.0
                D[t[i], t[j]] += area * np.dot(gi, gj) + (curv + m * m) * nn
                # T_vv' = int m (-N_v' dx N_v + N_v dx N_v')
                T[t[i], t[j]] += m * sum(-N(j, p) * np.dot(gi, east) + N(i, p) * np.dot(gj, east) for p in mids) * area / 3.0
    return D, T, A


def dense_from(m, vals):
    rp, col, _ = m.csr()
    M = np.zeros((m.nv, m.nv))
    for v in range(m.nv):
        M[v, col[rp[v]:rp[v + 1]]] = vals[rp[v]:rp[v + 1]]
    return M


@pytest.fixture(scope="module")
def band(oracle_mod):
    mesh = sphere_band(jitter_sphere(icosphere(2), 0.15, np.random.default_rng(5)), 62.0)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    m.build_vector(1.0)
    return mesh, m


def test_metric_matrices_match_their_definitions(band):
    mesh, m = band
    assert mesh.n_vert <= 300
    D, T, A = metric_matrices_by_quadrature(mesh.coords, mesh.tri, 1.0)
    dv, tv = m.vector_csr()
    Do, To = dense_from(m, dv), dense_from(m, tv)
    assert np.abs(Do - D).max() <= 1e-12 * np.abs(D).max()
    assert np.abs(To - T).max() <= 1e-12 * np.abs(T).max() and np.abs(T).max() > 1e-3
    assert np.abs(A - m.area()).max() <= 1e-13 * A.max()
    assert np.abs(To + To.T).max() <= 1e-14 and np.abs(np.diag(To)).max() == 0.0      # antisymmetric
    assert np.abs(Do - Do.T).max() <= 1e-14
    D2 = np.block([[Do, To], [-To, Do]])
    assert np.abs(D2 - D2.T).max() <= 1e-14                                           # hence D_2 symmetric
    assert np.linalg.eigvalsh(D2).min() >= -1e-12 * np.abs(D2).max()                  # and positive semidefinite


@pytest.mark.parametrize("n", [1, 2])
def test_vector_solve_against_dense_definition(band, n):
    mesh, m = band
    D, T, A = metric_matrices_by_quadrature(mesh.coords, mesh.tri, 1.0)
    D2 = np.block([[D, T], [-T, D]])
    M2 = np.concatenate([A, A])
    u, v = sphere_velocity_field(mesh.coords, 4, 12, np.random.default_rng(6))
    rng = np.random.default_rng(7)
    for ell in (0.5 * mesh.h, 2.0 * mesh.h, 5.0 * mesh.h):
        S2 = np.diag(M2) + GAMMA * ell ** (2 * n) * (D2 if n == 1 else D2 @ np.diag(1.0 / M2) @ D2)
        ref = np.linalg.solve(S2, M2 * np.concatenate([u, v]))
        xu, xv, info = m.solve_vector(u, v, ell, n)
        assert info["status"] == 0 and info["true_res"] <= 1e-10
        tol = max(1e-10, 20 * np.finfo(float).eps * np.linalg.cond(S2))
        assert np.linalg.norm(np.concatenate([xu, xv]) - ref) <= tol * np.linalg.norm(ref)
        pu, pv = rng.normal(size=mesh.n_vert), rng.normal(size=mesh.n_vert)
        ou, ov = m.apply_vector(pu, pv, ell, n)
        want = S2 @ np.concatenate([pu, pv])
        assert np.linalg.norm(np.concatenate([ou, ov]) - want) <= 1e-12 * np.linalg.norm(want)
    # first PCG iterate: exposes the Jacobi diagonal diag(S_2)
    ell = 2.0 * mesh.h
    S2 = np.diag(M2) + GAMMA * ell ** (2 * n) * (D2 if n == 1 else D2 @ np.diag(1.0 / M2) @ D2)
    phi = np.concatenate([u, v])
    r0 = M2 * phi - S2 @ phi
    z0 = r0 / np.diag(S2)
    alpha = (r0 @ z0) / (z0 @ (S2 @ z0))
    xu, xv, info = m.solve_vector(u, v, ell, n, max_iter=1)
    assert info["iters"] == 1
    assert np.linalg.norm(np.concatenate([xu, xv]) - (phi + alpha * z0)) <= 1e-11 * np.linalg.norm(phi)


@pytest.mark.parametrize("n", [1, 2])
def test_planar_mesh_has_no_metric_terms(oracle_mod, n):
    mesh = grid_mesh(10, periodic=True, jitter=0.2, random_diagonals=True, rng=np.random.default_rng(8))
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    m.build_vector()
    dv, tv = m.vector_csr()
    _, _, sv = m.csr()
    assert np.abs(tv).max() == 0.0 and np.abs(dv - sv).max() <= 1e-13 * np.abs(sv).max()
    rng = np.random.default_rng(9)
    u, v = rng.normal(size=mesh.n_vert), rng.normal(size=mesh.n_vert)
    for ell in (0.8, 3.0):
        xu, xv, info = m.solve_vector(u, v, ell, n)
        su, _ = m.solve(u, ell, n)
        sv_, _ = m.solve(v, ell, n)
        assert info["status"] == 0
        assert np.linalg.norm(xu - su) <= 1e-10 * np.linalg.norm(su) and np.linalg.norm(xv - sv_) <= 1e-10 * np.linalg.norm(sv_)


@pytest.mark.parametrize("axis", [(0.0, 0.0, 1.0), (1.0, 0.0, 0.0), (0.6, -0.8, 0.0)])
@pytest.mark.parametrize("n", [1, 2])
def test_rigid_rotation_is_attenuated_like_an_l1_harmonic(oracle_mod, axis, n):
    """U = a x x is a Killing field: rough Laplacian = Ricci = U / R^2, so the vector Laplacian of PAPER.md:89
    (grad.grad + R^-2, metric terms included) gives 2 U / R^2, and the filter multiplies U by 1 / (1 + gamma (2 l^2)^n)
    up to discretisation error and the boundary layer at the edges of the band.  l = 0.2: the attenuation differs from
    1 by 3.9e-2 (n = 1) / 3.2e-3 (n = 2); measured error of the coupled solve 1e-4 ... 5e-4 / 8e-4 ... 9e-4, of the same
    solve WITHOUT the coupling T (u and v as two scalars) 1.8e-2 ... 2.5e-2 / 9e-3.  (n = 2 about the polar axis is left
    out: there the biharmonic boundary layer of the band, 4e-3, exceeds the effect.)"""
    if n == 2 and abs(axis[2]) > 0.9:
        pytest.skip("boundary layer of the band exceeds the attenuation for this case")
    if n == 2 and axis[1] != 0.0:
        pytest.skip("n = 2 is checked about one equatorial axis (a minute of oracle time per axis)")
    mesh = sphere_band(jitter_sphere(icosphere(5), 0.15, np.random.default_rng(10)), 75.0)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    m.build_vector(1.0)
    a = np.array(axis) / np.linalg.norm(axis)
    U = np.cross(a[None, :], mesh.coords)
    east, north = sphere_frames(mesh.coords)
    u, v = np.einsum("ij,ij->i", U, east), np.einsum("ij,ij->i", U, north)
    ell = 0.2
    xu, xv, info = m.solve_vector(u, v, ell, n)
    assert info["status"] == 0
    g = 1.0 / (1.0 + GAMMA * (2.0 * ell ** 2) ** n)
    lat = np.degrees(np.arcsin(mesh.coords[:, 2]))
    inner = np.abs(lat) < 75.0 - np.degrees(3.5 * ell)
    err = np.hypot(xu - g * u, xv - g * v)[inner].max() / np.hypot(u, v).max()
    assert err <= (1e-3 if n == 1 else 1.5e-3), err
    su, _ = m.solve(u, ell, n)                                       # the same without the coupling
    sv, _ = m.solve(v, ell, n)
    err_scalar = np.hypot(su - g * u, sv - g * v)[inner].max() / np.hypot(u, v).max()
    assert err_scalar > (10 if n == 1 else 5) * err
