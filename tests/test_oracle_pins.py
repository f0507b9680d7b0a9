"""Pins of the CPU oracle against things other than itself (CPU only, no GPU).

Each test fixes the oracle to what the paper and the mathematics fix:
  * the definition S_vv' = integral grad N_v . grad N_v' dS with P1 basis functions,
    evaluated here from numerically inverted affine basis functions, not the cotangent closed form;
  * the median-dual control volume (PAPER.md:41 Fig. 1a, :47) measured as a polygon (shoelace);
  * "On uniform meshes (M^L)^-1 D~ = D": the 5-point stencil; the equilateral lattice;
  * plane waves on the uniform periodic grid are eigenvectors: attenuation 1/(1+gamma (l^2 lambda_k)^n)
    (BASELINE.json north_star; eq. (1));
  * dense direct solves by numpy.linalg (library routine) on meshes <= 500 vertices;
  * S symmetric, S 1 = 0, mean conservation, energy identity and monotonicity, limits in l;
  * Laplace-Beltrami eigenvalues l(l+1) on the unit icosphere.
A plausible slip anywhere (dropped term, sign, index, transposed operand) fails at least one of them.
"""
import numpy as np
import pytest

from workloads import equilateral_mesh, grid_mesh, icosphere, jitter_sphere, make_config

GAMMA = 0.5


# ---------------------------------------------------------------- definitions written out in the test
def p1_stiffness_and_dual_area(coords, tri, period=None):
    """Dense S and A_v straight from the definitions (no cotangents):
    N_i affine with N_i(x_j) = delta_ij on each flat triangle -> grad N_i from the inverse of [1 x y];
    S += area * grad N_i . grad N_j;  A_v += area of the quadrilateral vertex / mid-edge / centroid / mid-edge."""
    nv = coords.shape[0]
    S = np.zeros((nv, nv))
    A = np.zeros(nv)
    for t in tri:
        x0 = coords[t[0]]
        pts = [np.zeros_like(x0)]
        for k in (1, 2):
            d = coords[t[k]] - x0
            if period is not None:
                d = d - period * np.round(d / period)
            pts.append(d)
        # local orthonormal 2-D frame in the triangle's plane
        e1 = pts[1] / np.linalg.norm(pts[1])
        w = pts[2] - np.dot(pts[2], e1) * e1
        e2 = w / np.linalg.norm(w)
        q = np.array([[np.dot(p, e1), np.dot(p, e2)] for p in pts])
        B = np.linalg.inv(np.column_stack([np.ones(3), q]))   # columns: coefficients (a, gx, gy) of N_0..N_2
        G = B[1:, :].T                                         # [3][2] gradients
        area = 0.5 * abs(q[1, 0] * q[2, 1] - q[1, 1] * q[2, 0])
        S[np.ix_(t, t)] += area * (G @ G.T)
        cen = q.mean(axis=0)
        for i in range(3):
            a, b = q[(i + 1) % 3], q[(i + 2) % 3]
            poly = np.array([q[i], 0.5 * (q[i] + a), cen, 0.5 * (q[i] + b)])
            xs, ys = poly[:, 0], poly[:, 1]
            A[t[i]] += 0.5 * abs(np.dot(xs, np.roll(ys, -1)) - np.dot(ys, np.roll(xs, -1)))
    return S, A


def dense_from_csr(m):
    rp, col, val = m.csr()
    D = np.zeros((m.nv, m.nv))
    for v in range(m.nv):
        D[v, col[rp[v]:rp[v + 1]]] = val[rp[v]:rp[v + 1]]
    return D


def small_meshes():
    rng = np.random.default_rng(7)
    a = grid_mesh(8, periodic=True, jitter=0.25, random_diagonals=True, rng=rng)
    b = grid_mesh(7, periodic=False, jitter=0.2, random_diagonals=True, rng=rng)
    c = jitter_sphere(icosphere(2), 0.2, rng)
    return [a, b, c]


# ---------------------------------------------------------------- assembly
@pytest.mark.parametrize("idx", [0, 1, 2])
def test_assembly_matches_p1_definition(oracle_mod, idx):
    mesh = small_meshes()[idx]
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    S_def, A_def = p1_stiffness_and_dual_area(mesh.coords, mesh.tri, mesh.period)
    S = dense_from_csr(m)
    assert np.abs(S - S_def).max() <= 1e-12 * np.abs(S_def).max()
    assert np.abs(m.area() - A_def).max() <= 1e-13 * A_def.max()
    # structure: exactly the mesh edges plus the diagonal
    edges = set()
    for t in mesh.tri:
        for i in range(3):
            edges.add((int(t[i]), int(t[(i + 1) % 3])))
            edges.add((int(t[(i + 1) % 3]), int(t[i])))
    assert m.nnz == len(edges) + m.nv


def test_uniform_grid_is_five_point_stencil(oracle_mod):
    """on uniform meshes M^-1 S is the usual Laplacian; cells split along one diagonal give
    (4,-1,-1,-1,-1), the two diagonal-edge weights are exactly 0 (right angles), A_v = h^2."""
    n, h = 16, 0.5
    mesh = grid_mesh(n, periodic=True, h=h)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    S = dense_from_csr(m)
    assert np.allclose(m.area(), h * h, rtol=0, atol=1e-15)
    for v in (0, 5, n * n - 1, 37):
        ix, iy = v % n, v // n
        nb = [((ix + 1) % n) + iy * n, ((ix - 1) % n) + iy * n, ix + ((iy + 1) % n) * n, ix + ((iy - 1) % n) * n]
        dg = [((ix + 1) % n) + ((iy + 1) % n) * n, ((ix - 1) % n) + ((iy - 1) % n) * n]
        assert abs(S[v, v] - 4.0) < 1e-14
        assert np.allclose(S[v, nb], -1.0, atol=1e-14)
        assert np.allclose(S[v, dg], 0.0, atol=1e-15)
        assert abs(S[v].sum()) < 1e-14
    assert m.nnz == 7 * n * n


def test_equilateral_lattice(oracle_mod):
    mesh = equilateral_mesh(6, 6, h=2.0)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    rp, col, val = m.csr()
    assert np.allclose(m.area(), np.sqrt(3.0) / 2.0 * 4.0, rtol=1e-14)
    for v in range(m.nv):
        c, w = col[rp[v]:rp[v + 1]], val[rp[v]:rp[v + 1]]
        assert len(c) == 7
        assert np.allclose(w[c != v], -1.0 / np.sqrt(3.0), rtol=1e-13)
        assert np.isclose(w[c == v][0], 6.0 / np.sqrt(3.0), rtol=1e-13)


def test_symmetry_rowsums_total_area(oracle_mod):
    w = make_config(2, n=48)
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    S = dense_from_csr(m)
    assert np.abs(S - S.T).max() <= 1e-13 * np.abs(S).max()
    assert np.abs(S.sum(axis=1)).max() <= 1e-11 * np.abs(S).max()
    # milder jitter: no inverted triangles, so the dual areas tile the periodic square exactly
    mesh = grid_mesh(32, periodic=True, jitter=0.2, random_diagonals=True, rng=np.random.default_rng(3))
    m2 = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    assert abs(m2.area().sum() - 32.0 * 32.0) < 1e-9


def test_icosphere_area_converges_to_4pi(oracle_mod):
    deficits = []
    for L in (2, 3, 4):
        mesh = icosphere(L)
        m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
        assert m.nv == 10 * 4 ** L + 2 and mesh.n_tri == 20 * 4 ** L
        deficits.append(4.0 * np.pi - m.area().sum())
    assert all(d > 0 for d in deficits)                     # flat triangles lie inside the sphere
    assert 3.7 < deficits[0] / deficits[1] < 4.3 and 3.7 < deficits[1] / deficits[2] < 4.3


def test_p1_exactness_on_linear_functions(oracle_mod):
    """S (a.x) vanishes at interior vertices of a planar patch: P1 elements reproduce linear fields."""
    n = 9
    mesh = grid_mesh(n, periodic=False, jitter=0.25, random_diagonals=True, rng=np.random.default_rng(11))
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    f = 0.7 * mesh.coords[:, 0] - 1.3 * mesh.coords[:, 1] + 2.0
    y = m.apply_S(f)
    ix, iy = np.arange((n + 1) ** 2) % (n + 1), np.arange((n + 1) ** 2) // (n + 1)
    interior = (ix > 0) & (ix < n) & (iy > 0) & (iy < n)
    assert np.abs(y[interior]).max() < 1e-12
    assert np.abs(y[~interior]).max() > 1e-3                # boundary rows carry the (dropped) flux term


def test_icosphere_eigenvalues(oracle_mod):
    """Smallest eigenvalues of M^-1 S on the unit sphere approach l(l+1): 0, 2,2,2, 6 x5."""
    mesh = icosphere(3)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    S = dense_from_csr(m)
    a = m.area()
    K = S / np.sqrt(a)[:, None] / np.sqrt(a)[None, :]
    ev = np.linalg.eigvalsh(K)[:9]
    assert abs(ev[0]) < 1e-10
    assert np.allclose(ev[1:4], 2.0, rtol=2e-2)
    assert np.allclose(ev[4:9], 6.0, rtol=3e-2)


def test_error_paths(oracle_mod):
    coords = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [5.0, 5.0]])
    with pytest.raises(ValueError, match="no triangle"):
        oracle_mod.OracleMesh(coords, np.array([[0, 1, 2]], dtype=np.int32))
    with pytest.raises(ValueError, match="index"):
        oracle_mod.OracleMesh(coords[:3], np.array([[0, 1, 3]], dtype=np.int32))
    with pytest.raises(ValueError, match="index"):
        oracle_mod.OracleMesh(coords[:3], np.array([[0, 1, 1]], dtype=np.int32))
    flat = np.array([[0.0, 0.0], [1.0, 0.0], [2.0, 0.0]])
    with pytest.raises(ValueError, match="degenerate"):
        oracle_mod.OracleMesh(flat, np.array([[0, 1, 2]], dtype=np.int32))


# ---------------------------------------------------------------- operator and solve
@pytest.mark.parametrize("idx", [0, 1, 2])
@pytest.mark.parametrize("n", [1, 2])
def test_solve_against_definition_dense(oracle_mod, idx, n):
    """Whole chain on <= 500 vertices: S, A_v from the definitions above, A_l formed densely as written in
    PAPER.md:61 / :63, solved by numpy.linalg.solve; oracle CG and oracle Cholesky must both agree."""
    mesh = small_meshes()[idx]
    assert mesh.n_vert <= 500
    S, A = p1_stiffness_and_dual_area(mesh.coords, mesh.tri, mesh.period)
    rng = np.random.default_rng(100 + idx)
    phi = rng.normal(size=mesh.n_vert)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    for ell in (0.5 * mesh.h, 2.0 * mesh.h, 6.0 * mesh.h):
        if n == 1:
            Al = np.diag(A) + GAMMA * ell ** 2 * S
        else:
            Al = np.diag(A) + GAMMA * ell ** 4 * S @ np.diag(1.0 / A) @ S
        ref = np.linalg.solve(Al, A * phi)
        x, info = m.solve(phi, ell, n)
        assert info["status"] == 0
        assert np.linalg.norm(x - ref) <= 1e-10 * np.linalg.norm(ref)
        xd = m.dense_solve(phi, ell, n)
        assert np.linalg.norm(xd - ref) <= 1e-11 * np.linalg.norm(ref)
        # operator itself
        p = rng.normal(size=mesh.n_vert)
        assert np.linalg.norm(m.apply(p, ell, n) - Al @ p) <= 1e-12 * np.linalg.norm(Al @ p)


@pytest.mark.parametrize("n", [1, 2])
def test_config1_closed_form(oracle_mod, n):
    """Config 1: every lattice plane wave is an eigenvector of the 5-point Laplacian with
    lambda_m = (4 - 2cos(2 pi m_x/N) - 2cos(2 pi m_y/N))/h^2, so
    phibar = sum_j a_j cos(.)/(1 + gamma (l^2 lambda_mj)^n) exactly (north_star pin 3)."""
    w = make_config(1)
    N = 64
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    wv = w.waves[0]
    lam = 4.0 - 2.0 * np.cos(2 * np.pi * wv.k[:, 0] / N) - 2.0 * np.cos(2 * np.pi * wv.k[:, 1] / N)
    basis = np.cos(w.mesh.coords @ (wv.k.T * wv.scale) + wv.theta)
    assert np.linalg.norm(basis @ wv.amp - w.fields[0]) <= 1e-13 * np.linalg.norm(w.fields[0])
    ells = w.ells if n == 1 else w.ells[w.ells <= 8.0]
    for ell in ells:
        g = 1.0 / (1.0 + GAMMA * (ell ** 2 * lam) ** n)
        ref = basis @ (wv.amp * g)
        x, info = m.solve(w.fields[0], ell, n)
        assert info["status"] == 0
        assert np.linalg.norm(x - ref) <= 2e-12 * np.linalg.norm(ref)
        # energy of the closed form (A_v = 1: plain mean)
        assert abs(m.energy(x) - 0.5 * np.mean(ref ** 2)) <= 1e-11 * 0.5 * np.mean(ref ** 2)


def test_medium_mesh_against_sparse_direct(oracle_mod):
    """Config-2-like sliver mesh, 64^2: oracle CG against SciPy's sparse LU of the explicitly formed system."""
    sp = pytest.importorskip("scipy.sparse")
    spla = pytest.importorskip("scipy.sparse.linalg")
    w = make_config(2, n=64)
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    rp, col, val = m.csr()
    S = sp.csr_matrix((val, col, rp), shape=(m.nv, m.nv))
    A = m.area()
    for n, ell in ((1, 1.0), (1, 8.0), (1, 32.0), (2, 2.0)):
        if n == 1:
            Al = sp.diags(A) + GAMMA * ell ** 2 * S
        else:
            Al = sp.diags(A) + GAMMA * ell ** 4 * (S @ sp.diags(1.0 / A) @ S)
        ref = spla.spsolve(Al.tocsc(), A * w.fields[0])
        x, info = m.solve(w.fields[0], ell, n)
        assert info["status"] == 0
        assert np.linalg.norm(x - ref) <= 1e-9 * np.linalg.norm(ref)


def test_invariants_and_limits(oracle_mod):
    w = make_config(4, level=4, n_fields=1)
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    A = m.area()
    phi = w.fields[0] + 0.3
    mean = np.dot(A, phi) / A.sum()
    prev = None
    for n in (1, 2):
        prev = None
        for ell in w.mesh.h * np.array([0.25, 1.0, 3.0, 9.0]):
            x, info = m.solve(phi, ell, n)
            assert info["status"] == 0
            # S 1 = 0 and S symmetric: the area-weighted mean is conserved (north_star pin 2)
            assert abs(np.dot(A, x) - np.dot(A, phi)) <= 1e-11 * np.abs(A * phi).sum()
            # energy identity phi^T M x = x^T A_l x >= x^T M x
            lhs = np.dot(A * phi, x)
            rhs = np.dot(x, m.apply(x, ell, n))
            assert abs(lhs - rhs) <= 1e-10 * abs(lhs)
            assert rhs >= np.dot(A * x, x) * (1 - 1e-12)
            # <phibar^2> monotone non-increasing in l (north_star pin 4)
            e = m.energy(x)
            if prev is not None:
                assert e <= prev * (1 + 1e-12)
            prev = e
    # limits: l -> 0 gives phi, l -> infinity gives the area-weighted mean (one connected component here)
    x0, _ = m.solve(phi, 1e-4 * w.mesh.h, 1)
    assert np.linalg.norm(x0 - phi) <= 1e-6 * np.linalg.norm(phi)
    xinf, info = m.solve(phi, 1e4, 1)
    assert np.abs(xinf - mean).max() <= 1e-6 * abs(mean)


def test_sphere_harmonic_attenuation(oracle_mod):
    """z on the unjittered unit icosphere is (to O(h^2)) the l=1 harmonic: attenuated by 1/(1+gamma (2 l^2)^n)."""
    mesh = icosphere(4)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    z = mesh.coords[:, 2].copy()
    for n, ell in ((1, 0.5), (2, 0.6)):
        x, _ = m.solve(z, ell, n)
        g = 1.0 / (1.0 + GAMMA * (2.0 * ell ** 2) ** n)
        assert np.linalg.norm(x - g * z) <= 2e-2 * np.linalg.norm(g * z)


# ---------------------------------------------------------------- energy and spectrum
def test_spectrum_hand_example(oracle_mod):
    """ells = 1, 2, 4 -> k = 1, 1/2, 1/4 (PAPER.md:35 k_l = 1/l); e = 3, 2, 1/2:
    E_0 = (3-2)/(1-1/2) = 2, E_1 = (2-1/2)/(1/2-1/4) = 6; k_mid = sqrt(1/2), sqrt(1/8)."""
    k_mid, E = oracle_mod.spectrum(np.array([1.0, 2.0, 4.0]), np.array([3.0, 2.0, 0.5]))
    assert np.allclose(E, [2.0, 6.0], rtol=1e-15)
    assert np.allclose(k_mid, [np.sqrt(0.5), np.sqrt(0.125)], rtol=1e-15)


def test_energy_definition(oracle_mod):
    mesh = small_meshes()[1]
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    _, A = p1_stiffness_and_dual_area(mesh.coords, mesh.tri, None)
    x = np.random.default_rng(5).normal(size=mesh.n_vert)
    assert abs(m.energy(x) - 0.5 * np.sum(A * x * x) / np.sum(A)) <= 1e-14 * m.energy(x)


def test_spectrum_properties(oracle_mod):
    w = make_config(2, n=48, n_ells=8, ell_max=16.0)
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out, en, k_mid, E, infos = oracle_mod.filter_and_spectrum(m, w.fields, w.ells, 1)
    assert all(i["status"] == 0 for row in infos for i in row)
    k = 1.0 / w.ells
    for f in range(w.fields.shape[0]):
        assert np.all(np.diff(en[f]) <= 0)                                     # monotone
        assert np.all(E[f] >= 0)
        assert abs(np.sum(E[f] * (k[:-1] - k[1:])) - (en[f, 0] - en[f, -1])) <= 1e-13 * en[f, 0]   # telescoping
    assert np.allclose(k_mid, np.sqrt(k[:-1] * k[1:]), rtol=1e-15)


def test_golden_config1(oracle_mod):
    """tests/golden/config1_closed_form.txt holds closed-form (not solver) energies of config 1, written by
    tests/golden/make_golden.py from the plane-wave attenuation formula; the oracle must reproduce them."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "config1_closed_form.txt")
    rows = np.loadtxt(path, comments="#")
    w = make_config(1)
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    assert np.allclose(rows[:, 0], w.ells, rtol=1e-14)
    for ell, e_ref in rows:
        x, _ = m.solve(w.fields[0], ell, 1)
        assert abs(m.energy(x) - e_ref) <= 1e-11 * e_ref


# ---------------------------------------------------------------- higher orders n = 3, 4
@pytest.mark.parametrize("idx", [0, 1, 2])
@pytest.mark.parametrize("n", [3, 4])
def test_higher_order_against_definition_dense(oracle_mod, idx, n):
    """"This procedure can be generalized to higher-order filters": A_l = M + gamma l^(2n) S (M^-1 S)^(n-1),
    formed densely from the P1 definitions (not from the oracle's assembly) and solved by numpy; the oracle's
    operator, its Jacobi-PCG, its dense Cholesky path and the Jacobi diagonal it builds must agree with it."""
    mesh = small_meshes()[idx]
    S, A = p1_stiffness_and_dual_area(mesh.coords, mesh.tri, mesh.period)
    rng = np.random.default_rng(300 + 10 * idx + n)
    phi = rng.normal(size=mesh.n_vert)
    m = oracle_mod.OracleMesh(mesh.coords, mesh.tri, mesh.period)
    MiS = S / A[:, None]
    for ell in (0.5 * mesh.h, 1.5 * mesh.h, 3.0 * mesh.h):
        Al = np.diag(A) + GAMMA * ell ** (2 * n) * S @ np.linalg.matrix_power(MiS, n - 1)
        assert np.abs(Al - Al.T).max() <= 1e-10 * np.abs(Al).max()           # symmetric, as PAPER.md:61 states for n = 1
        ref = np.linalg.solve(Al, A * phi)
        # fp64 floor of ANY solve of this system, the numpy reference included: a few u cond(A_l) (cond reaches 5e8 for
        # n = 4 at 3 h -- the reason reading A16-like ranges bound the higher orders)
        tol = max(1e-10, 20.0 * np.finfo(float).eps * np.linalg.cond(Al))
        x, info = m.solve(phi, ell, n)
        assert info["status"] == 0
        assert np.linalg.norm(x - ref) <= tol * np.linalg.norm(ref)
        xd = m.dense_solve(phi, ell, n)
        assert np.linalg.norm(xd - ref) <= tol * np.linalg.norm(ref)
        p = rng.normal(size=mesh.n_vert)
        assert np.linalg.norm(m.apply(p, ell, n) - Al @ p) <= 1e-12 * np.linalg.norm(Al @ p)
    # the Jacobi diagonal: one PCG step from x0 = 0-like data exposes d only through the iterates, so check it through
    # the first iterate of a solve with max_iter = 1: x1 = phi + alpha z0, z0 = r0 / d
    ell = 1.5 * mesh.h
    Al = np.diag(A) + GAMMA * ell ** (2 * n) * S @ np.linalg.matrix_power(MiS, n - 1)
    r0 = A * phi - Al @ phi
    z0 = r0 / np.diag(Al)
    alpha = (r0 @ z0) / (z0 @ (Al @ z0))
    x1, info = m.solve(phi, ell, n, max_iter=1)
    assert info["iters"] == 1 and np.linalg.norm(x1 - (phi + alpha * z0)) <= 1e-11 * np.linalg.norm(x1)


@pytest.mark.parametrize("n", [3, 4])
def test_config1_closed_form_higher_order(oracle_mod, n):
    """The plane-wave attenuation 1 / (1 + gamma (l^2 lambda_m)^n) on config 1 holds for every order n."""
    w = make_config(1)
    N = 64
    m = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    wv = w.waves[0]
    lam = 4.0 - 2.0 * np.cos(2 * np.pi * wv.k[:, 0] / N) - 2.0 * np.cos(2 * np.pi * wv.k[:, 1] / N)
    basis = np.cos(w.mesh.coords @ (wv.k.T * wv.scale) + wv.theta)
    for ell in (1.0, 2.2) if n == 4 else (1.0, 3.0):
        g = 1.0 / (1.0 + GAMMA * (ell ** 2 * lam) ** n)
        ref = basis @ (wv.amp * g)
        x, info = m.solve(w.fields[0], ell, n)
        assert info["status"] == 0
        assert np.linalg.norm(x - ref) <= 1e-10 * np.linalg.norm(ref)
