"""GPU parity: the CUDA path, called through the C ABI (paper_2404_07398_b200.binding -> libimplicit_filter.so),
against the CPU oracle, element by element on the same seeded inputs.

Tolerances (BASELINE.json north_star): relative L2 <= 1e-7 per filtered field, <= 1e-6 per spectrum bin.
Assembly (integer structure) is compared exactly; fp64 values of S, A_v and of the operator to 1e-12, which is
the rounding of differently ordered sums of <= 10 terms ("tolerances").
"""
import numpy as np
import pytest

from workloads import grid_mesh, make_config

pytestmark = pytest.mark.gpu

TOL_FIELD = 1e-7
TOL_BIN = 1e-6


@pytest.fixture(scope="module")
def ifl():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2404_07398_b200 as lib
    lib.load_library()          # fails loudly if the extension is missing
    return lib


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(np.asarray(b)), 1e-300))


SMALL = {
    "cfg1": lambda: make_config(1),
    "cfg2_n96": lambda: make_config(2, n=96, n_ells=6, ell_max=24.0),
    "cfg3_L4": lambda: make_config(3, level=4, n_ells=5, ell_max=6.0),
    "cfg4_L5": lambda: make_config(4, level=5, n_ells=7),
    "cfg5_L4": lambda: make_config(5, level=4, n_fields=3, n_ells=4, ell_max=5.0),
}


# ------------------------------------------------------------------------------------------ preparation
@pytest.mark.parametrize("name", list(SMALL))
def test_prepare_matches_oracle_assembly(ifl, oracle_mod, name):
    w = SMALL[name]()
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period, flags=ifl.IF_FLAG_KEEP_CSR)
    rp, col, val, area = ifl.if_mesh_export_csr(h)
    orp, ocol, oval = om.csr()
    assert h.n_vert == om.nv and h.nnz == om.nnz
    assert np.array_equal(rp, orp)                      # bit-exact structure
    assert np.array_equal(col, ocol)
    assert np.abs(val - oval).max() <= 1e-12 * np.abs(oval).max()
    assert np.abs(area - om.area()).max() <= 1e-13 * om.area().max()
    assert abs(h.total_area - om.area().sum()) <= 1e-12 * om.area().sum()
    perm = ifl.if_mesh_export_perm(h)
    assert np.array_equal(np.sort(perm), np.arange(om.nv))
    assert h.sell_slots >= h.nnz - h.n_vert and h.sell_slots % 2 == 0
    h.close()


@pytest.mark.parametrize("opts", [dict(sfc_kind=1), dict(sell_sigma=32), dict(sell_c=64, sell_sigma=512),
                                  dict(sell_c=128, sell_sigma=128)])
def test_layout_options_do_not_change_results(ifl, oracle_mod, opts):
    w = SMALL["cfg4_L5"]()
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, **opts)
    ells = w.ells[[0, 3]]
    out = ifl.if_apply(h, w.fields, ells, 1).cpu().numpy()
    for f in range(w.fields.shape[0]):
        for j, ell in enumerate(ells):
            assert rel(out[f, j], om.apply(w.fields[f], ell, 1)) <= 1e-12
    h.close()


def test_prepare_error_codes(ifl):
    coords = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [5.0, 5.0]])
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_prepare(coords, np.array([[0, 1, 2]], dtype=np.int32))
    assert e.value.code == -4                                        # orphan vertex 3
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_prepare(coords[:3], np.array([[0, 1, 3]], dtype=np.int32))
    assert e.value.code == -2
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_prepare(coords[:3], np.array([[0, 1, 1]], dtype=np.int32))
    assert e.value.code == -2
    flat = np.array([[0.0, 0.0], [1.0, 0.0], [2.0, 0.0]])
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_prepare(flat, np.array([[0, 1, 2]], dtype=np.int32))
    assert e.value.code == -3
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_prepare(coords[:3], np.array([[0, 1, 2]], dtype=np.int32), sell_c=48)
    assert e.value.code == -1


# ------------------------------------------------------------------------------------------ operator (SpMM)
@pytest.mark.parametrize("name", list(SMALL))
@pytest.mark.parametrize("order_n", [1, 2])
def test_apply_matches_oracle_operator(ifl, oracle_mod, name, order_n):
    w = SMALL[name]()
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out = ifl.if_apply(h, w.fields, w.ells, order_n).cpu().numpy()
    for f in range(w.fields.shape[0]):
        for j, ell in enumerate(w.ells):
            assert rel(out[f, j], om.apply(w.fields[f], ell, order_n)) <= 1e-12, (f, j)
    h.close()


# ------------------------------------------------------------------------------------------ filter + spectrum
def check_workload(ifl, oracle_mod, w, order_n=None, **options):
    order_n = w.order_n if order_n is None else order_n
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    ref, en, k_mid, E, infos = oracle_mod.filter_and_spectrum(om, w.fields, w.ells, order_n)
    assert all(i["status"] == 0 for row in infos for i in row)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out, st = ifl.if_filter(h, w.fields, w.ells, order_n, **options)
    out = out.cpu().numpy()
    assert st["code"] == 0 and np.all(st["status"] == 0)
    for f in range(w.fields.shape[0]):
        for j in range(w.ells.shape[0]):
            assert rel(out[f, j], ref[f, j]) <= TOL_FIELD, (f, j, rel(out[f, j], ref[f, j]))
    sp = ifl.if_spectrum(h, w.fields, w.ells, order_n, **options)
    assert sp["stats"]["code"] == 0
    assert np.abs(sp["energy"] - en).max() <= TOL_BIN * np.abs(en).max()
    assert np.all(np.abs(sp["E"] - E) <= TOL_BIN * np.abs(E)), np.abs(sp["E"] / E - 1).max()
    assert np.allclose(sp["k_mid"], k_mid, rtol=1e-14)
    h.close()
    return out, sp, st


@pytest.mark.parametrize("name", list(SMALL))
def test_filter_and_spectrum_match_oracle(ifl, oracle_mod, name):
    check_workload(ifl, oracle_mod, SMALL[name]())


def test_config1_closed_form_on_gpu(ifl):
    """Config 1 against the plane-wave closed form directly (no oracle in between), and the golden energies."""
    import os
    w = make_config(1)
    N = 64
    wv = w.waves[0]
    lam = 4.0 - 2.0 * np.cos(2 * np.pi * wv.k[:, 0] / N) - 2.0 * np.cos(2 * np.pi * wv.k[:, 1] / N)
    basis = np.cos(w.mesh.coords @ (wv.k.T * wv.scale) + wv.theta)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out, st = ifl.if_filter(h, w.fields, w.ells, 1)
    out = out.cpu().numpy()
    for j, ell in enumerate(w.ells):
        ref = basis @ (wv.amp / (1.0 + 0.5 * ell ** 2 * lam))
        assert rel(out[0, j], ref) <= TOL_FIELD
    sp = ifl.if_spectrum(h, w.fields, w.ells, 1)
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "config1_closed_form.txt"), comments="#")
    assert np.abs(sp["energy"][0] - gold[:, 1]).max() <= TOL_BIN * gold[:, 1].max()
    h.close()


@pytest.mark.parametrize("batch", [4, 8, 16])
@pytest.mark.parametrize("n_ells", [1, 5, 9])
def test_batch_sizes_and_ragged_tails(ifl, oracle_mod, batch, n_ells):
    """R = 2 fields x n_ells right-hand sides never fills the last batch: unused columns must stay inert."""
    w = make_config(2, n=48, n_ells=max(n_ells, 2), ell_max=12.0)
    w.ells = w.ells[:n_ells] if n_ells > 1 else w.ells[1:2]
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out, st = ifl.if_filter(h, w.fields, w.ells, 1, batch=batch)
    out = out.cpu().numpy()
    for f in range(2):
        for j, ell in enumerate(w.ells):
            x, _ = om.solve(w.fields[f], ell, 1)
            assert rel(out[f, j], x) <= TOL_FIELD
    h.close()


def test_degenerate_inputs(ifl, oracle_mod):
    w = make_config(4, level=4, n_fields=1, n_ells=3)
    V = w.mesh.n_vert
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    fields = np.stack([np.full(V, 2.5), np.zeros(V), w.fields[0]])
    out, st = ifl.if_filter(h, fields, w.ells, 1)
    out = out.cpu().numpy()
    assert st["code"] == 0
    assert np.all(st["iters"][0] <= 1) and np.all(st["iters"][1] == 0)
    assert np.abs(out[0] - 2.5).max() <= 1e-12            # constants are fixed points (S 1 = 0)
    assert np.all(out[1] == 0.0)
    # iteration cap: a status, not a hang (convergence may be lost)
    out2, st2 = ifl.if_filter(h, w.fields, w.ells[-1:], 2, max_iter=4, check_every=2)
    assert st2["code"] == 1 and st2["status"][0, 0] == 1 and st2["iters"][0, 0] == 4
    assert np.all(np.isfinite(out2.cpu().numpy()))
    # argument errors
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h, w.fields, [1.0, -1.0], 1)
    assert e.value.code == -1
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h, w.fields, [1.0], 5)                     # orders 1 ... 4 exist
    assert e.value.code == -1
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_spectrum(h, w.fields, [2.0, 1.0], 1)
    assert e.value.code == -1
    import torch
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h, w.fields, [1.0], 1, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.code == -7
    # empty inputs and the largest job the result arrays serve (65 536 right-hand sides per call)
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h, w.fields, [], 1)
    assert e.value.code == -1
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_spectrum(h, w.fields, [1.0], 1)                   # a spectrum needs two scales
    assert e.value.code == -1
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_spectrum(h, w.fields, np.linspace(1.0, 2.0, 65537) * w.mesh.h, 1)
    assert e.value.code == -1
    for bad in (np.nan, np.inf, 0.0):
        with pytest.raises(ifl.ImplicitFilterError) as e:
            ifl.if_filter(h, w.fields, [1.0, bad], 1)
        assert e.value.code == -1
    h.close()


def test_tolerance_and_paper_setting(ifl, oracle_mod):
    """tol = 1e-9 stops earlier than the default and still lands within 1e-6 of the oracle."""
    w = make_config(2, n=64, n_ells=3, ell_max=16.0)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    o9, s9 = ifl.if_filter(h, w.fields[:1], w.ells, 1, tol=1e-9)
    o12, s12 = ifl.if_filter(h, w.fields[:1], w.ells, 1)
    assert np.all(s9["iters"] <= s12["iters"]) and s9["iters"].sum() < s12["iters"].sum()
    assert np.all(s12["rel_res"] <= 1e-12) and np.all(s9["rel_res"] <= 1e-9)
    for j, ell in enumerate(w.ells):
        x, _ = om.solve(w.fields[0], ell, 1)
        assert rel(o9[0, j].cpu().numpy(), x) <= 1e-6
    h.close()


def test_spectrum_from_host_buffers(ifl, oracle_mod):
    """if_spectrum_host: fields in host memory, copied inside the C call; same numbers as the device-pointer call."""
    import torch
    w = make_config(4, level=5, n_ells=7)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    a = ifl.if_spectrum(h, w.fields, w.ells, 1)
    pinned = torch.from_numpy(w.fields).pin_memory()
    b = ifl.if_spectrum_host(h, pinned, w.ells, 1)
    c = ifl.if_spectrum_host(h, w.fields, w.ells, 1)                     # pageable numpy memory works too
    assert b["stats"]["code"] == 0 and np.array_equal(a["energy"], b["energy"]) and np.array_equal(a["E"], c["E"])
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_spectrum_host(h, pinned, w.ells, 1, workspace=torch.empty(ifl.if_workspace_bytes(h, 1), dtype=torch.uint8,
                                                                         device="cuda"))
    assert e.value.code == -7                                            # no room for the fields in the workspace
    h.close()


def test_highpass_output(ifl, oracle_mod):
    """IF_FLAG_HIGHPASS: if_filter returns phi - phibar_l (Fig. 3)."""
    w = make_config(4, level=5, n_ells=5)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    hp, st = ifl.if_filter(h, w.fields, w.ells, 1, flags=ifl.IF_FLAG_HIGHPASS)
    lp, _ = ifl.if_filter(h, w.fields, w.ells, 1)                      # the flag is per call
    hp, lp = hp.cpu().numpy(), lp.cpu().numpy()
    assert st["code"] == 0
    for f in range(2):
        for j, ell in enumerate(w.ells):
            x, _ = om.solve(w.fields[f], ell, 1)
            assert rel(hp[f, j], w.fields[f] - x) <= TOL_FIELD
            assert rel(lp[f, j], x) <= TOL_FIELD
    h.close()


def test_save_and_load_prepared_mesh(ifl, tmp_path):
    """The prepared mesh is scale-independent and reusable from disk: bit-identical results."""
    w = make_config(3, level=4, n_ells=4, ell_max=4.0)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    a, _ = ifl.if_filter(h, w.fields, w.ells, 2)
    path = str(tmp_path / "mesh.ifm")
    ifl.if_save(h, path)
    h.close()
    g = ifl.if_load(path)
    assert (g.n_vert, g.n_tiles) == (w.mesh.n_vert, (w.mesh.n_vert + 127) // 128)
    b, st = ifl.if_filter(g, w.fields, w.ells, 2)
    assert st["code"] == 0 and bool((a == b).all())
    assert np.array_equal(np.sort(ifl.if_mesh_export_perm(g)), np.arange(w.mesh.n_vert))
    g.close()
    with open(path, "r+b") as fh:
        fh.write(b"garbage!")
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_load(path)
    assert e.value.code == -8
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_load(str(tmp_path / "missing.ifm"))
    assert e.value.code == -8


@pytest.mark.parametrize("n,periodic", [(8, True), (5, False), (12, False)])
def test_meshes_smaller_than_one_row_tile(ifl, oracle_mod, n, periodic):
    """Fewer vertices than one 128-row SpMM tile (64, 36, 169 with a ragged second tile): the persistent kernels
    see one or two tiles, most CTAs none; dense direct solve as the reference for the smallest."""
    m = grid_mesh(n, periodic=periodic, jitter=0.2, random_diagonals=True, rng=np.random.default_rng(n))
    rng = np.random.default_rng(100 + n)
    fields = rng.standard_normal((3, m.n_vert))
    ells = np.array([0.7, 2.0, 5.0])
    om = oracle_mod.OracleMesh(m.coords, m.tri, m.period)
    h = ifl.if_prepare(m.coords, m.tri, m.period)
    assert h.n_tiles == (m.n_vert + 127) // 128
    for order_n in (1, 2):
        out, st = ifl.if_filter(h, fields, ells, order_n)
        out = out.cpu().numpy()
        assert st["code"] == 0
        for f in range(3):
            for j, ell in enumerate(ells):
                ref = om.dense_solve(fields[f], ell, order_n) if m.n_vert <= 500 else om.solve(fields[f], ell, order_n)[0]
                assert rel(out[f, j], ref) <= TOL_FIELD, (order_n, f, j)
    h.close()


# ------------------------------------------------------------------------------------------ multigrid-preconditioned CG
@pytest.mark.parametrize("name", ["cfg1", "cfg2_n96", "cfg4_L5"])
def test_multigrid_solver_matches_oracle(ifl, oracle_mod, name):
    """solver = 1: the large scales go through the smoothed-aggregation V-cycle PCG, the small ones through
    Jacobi-PCG; same systems, same answers (1e-7 per field, 1e-6 per bin), far fewer iterations at large l."""
    w = SMALL[name]()
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    ref, en, k_mid, E, _ = oracle_mod.filter_and_spectrum(om, w.fields, w.ells, 1)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period, flags=ifl.IF_FLAG_MULTIGRID)
    out, st = ifl.if_filter(h, w.fields, w.ells, 1, solver=1, mg_min_ell=2.0)
    jac, stj = ifl.if_filter(h, w.fields, w.ells, 1)
    out = out.cpu().numpy()
    assert st["code"] == 0 and np.all(st["rel_res"] <= 1e-12)
    for f in range(w.fields.shape[0]):
        for j in range(w.ells.shape[0]):
            assert rel(out[f, j], ref[f, j]) <= TOL_FIELD, (f, j)
    big = w.ells >= 2.0 * h.mean_edge
    assert big.any() and st["iters"][:, big].sum() < stj["iters"][:, big].sum()
    # small scales take the Jacobi path (another column width may move a stop by an iteration)
    assert np.abs(st["iters"][:, ~big] - stj["iters"][:, ~big]).max(initial=0) <= 2
    sp = ifl.if_spectrum(h, w.fields, w.ells, 1, solver=1, mg_min_ell=2.0)
    assert np.all(np.abs(sp["E"] - E) <= TOL_BIN * np.abs(E))
    h.close()


def test_multigrid_option_is_ignored_where_it_does_not_apply(ifl, oracle_mod):
    """A handle without hierarchy, or a narrower batch: solver = 1 silently means Jacobi-PCG; solver = 2 asks for
    Jacobi-PCG on a handle whose default is multigrid."""
    w = SMALL["cfg4_L5"]()
    h0 = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    h1 = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    a, sa = ifl.if_filter(h0, w.fields, w.ells, 1)
    for h, kw in ((h0, dict(solver=1)), (h1, dict(solver=1, batch=8))):
        b, sb = ifl.if_filter(h, w.fields, w.ells, 1, **kw)
        assert np.abs(sa["iters"] - sb["iters"]).max() <= 2
        assert float((a - b).abs().max()) <= 1e-9 * float(a.abs().max())
    h2 = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID, solver=1)
    c, sc = ifl.if_filter(h2, w.fields, w.ells, 1)              # the handle's default: multigrid
    d, sd = ifl.if_filter(h2, w.fields, w.ells, 1, solver=2)    # explicitly Jacobi
    assert sc["iters"].sum() < 0.5 * sa["iters"].sum() and np.abs(sd["iters"] - sa["iters"]).max() <= 2
    h0.close(); h1.close(); h2.close()


def test_multigrid_on_disconnected_and_degenerate_inputs(ifl, oracle_mod):
    """Three components (two jittered 40 x 40 grids and a lone triangle), scales far above their size: the filter
    tends to each component's own area-weighted mean, which the graph aggregates must respect.  Also constants and
    zeros (no iteration), the iteration cap (a status), high-pass output and host buffers with solver = 1."""
    a = grid_mesh(40, periodic=False, jitter=0.25, random_diagonals=True, rng=np.random.default_rng(5))
    b = grid_mesh(40, periodic=False, jitter=0.25, random_diagonals=True, rng=np.random.default_rng(6))
    lone = np.array([[200.0, 0.0], [201.0, 0.1], [200.4, 0.9]])
    coords = np.concatenate([a.coords, b.coords + np.array([60.0, 3.0]), lone])
    tri = np.concatenate([a.tri, b.tri + a.n_vert, np.array([[0, 1, 2]], dtype=np.int32) + 2 * a.n_vert]).astype(np.int32)
    V = coords.shape[0]
    rng = np.random.default_rng(77)
    fields = np.stack([rng.standard_normal(V), np.full(V, -1.5), np.zeros(V)])
    ells = np.array([1.0, 6.0, 40.0, 400.0])
    om = oracle_mod.OracleMesh(coords, tri, None)
    h = ifl.if_prepare(coords, tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    out, st = ifl.if_filter(h, fields, ells, 1, solver=1, mg_min_ell=2.0)
    jac, stj = ifl.if_filter(h, fields, ells, 1)
    out = out.cpu().numpy()
    assert st["code"] == 0 and np.all(st["rel_res"] <= 1e-12)
    for j, ell in enumerate(ells):
        x, info = om.solve(fields[0], float(ell), 1)
        assert info["status"] == 0 and rel(out[0, j], x) <= TOL_FIELD, j
    assert st["iters"][0, 1:].max() < 80 and stj["iters"][0, 3] > 10 * st["iters"][0, 3]
    area = om.area()
    for lo, hi in ((0, a.n_vert), (a.n_vert, 2 * a.n_vert), (2 * a.n_vert, V)):      # per-component means at l = 400
        mean = float((area[lo:hi] * fields[0, lo:hi]).sum() / area[lo:hi].sum())
        assert np.abs(out[0, 3, lo:hi] - mean).max() <= 2e-2 * np.abs(fields[0]).max()
        assert abs(float((area[lo:hi] * out[0, 3, lo:hi]).sum() / area[lo:hi].sum()) - mean) <= 1e-10
    # a constant is a fixed point (S 1 = 0): nothing to do but to clean up the rounding of c S 1 at l = 400
    assert np.all(st["iters"][1, :3] <= 1) and st["iters"][1, 3] <= 8 and np.all(st["iters"][2] == 0)
    assert np.abs(out[1] + 1.5).max() <= 1e-9 and np.all(out[2] == 0.0)     # (the lone triangle is the loosest)
    # iteration cap inside the multigrid path
    o2, s2 = ifl.if_filter(h, fields[:1], ells[-1:], 1, solver=1, mg_min_ell=2.0, max_iter=3)
    assert s2["code"] == 1 and s2["status"][0, 0] == 1 and s2["iters"][0, 0] == 3
    assert np.all(np.isfinite(o2.cpu().numpy()))
    # high-pass output and host buffers
    hp, _ = ifl.if_filter(h, fields[:1], ells, 1, solver=1, mg_min_ell=2.0, flags=ifl.IF_FLAG_HIGHPASS)
    assert rel(hp[0].cpu().numpy(), fields[0][None, :] - out[0]) <= 1e-10
    sp_d = ifl.if_spectrum(h, fields[:1], ells, 1, solver=1, mg_min_ell=2.0)
    sp_h = ifl.if_spectrum_host(h, fields[:1], ells, 1, solver=1, mg_min_ell=2.0)
    assert np.array_equal(sp_d["energy"], sp_h["energy"])
    en = np.array([om.energy(om.solve(fields[0], float(l), 1)[0]) for l in ells])
    assert np.all(np.abs(sp_d["energy"][0] - en) <= TOL_BIN * en)
    h.close()


def test_multigrid_fused_residual_kernel_on_unstaged_tiles(ifl, oracle_mod):
    """k_spmm<16, MGR> (r' = r - alpha q, e = omega r'/d, t = r' - A e in one pass) has two gather paths: tiles whose
    halo fits the shared-memory stage and tiles that read their out-of-tile rows from global memory.  A shuffled
    vertex order kept as it is (sfc_kind = 1) makes every tile of the second kind; both orders must give the oracle's
    fields, and the iteration counts may differ only by what another summation order moves a stop."""
    w = SMALL["cfg4_L5"]()
    V = w.mesh.n_vert
    rng = np.random.default_rng(11)
    new_of_old = rng.permutation(V)
    coords = np.empty_like(w.mesh.coords)
    coords[new_of_old] = w.mesh.coords
    tri = new_of_old[w.mesh.tri].astype(np.int32)
    fields = np.empty_like(w.fields)
    fields[:, new_of_old] = w.fields
    ells = w.ells[-3:]
    om = oracle_mod.OracleMesh(coords, tri, None)
    h_sfc = ifl.if_prepare(coords, tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    h_raw = ifl.if_prepare(coords, tri, None, flags=ifl.IF_FLAG_MULTIGRID, sfc_kind=1)
    # (the ragged last tile has few rows and may still fit)
    assert h_raw.unstaged_tiles >= h_raw.n_tiles - 1 and h_sfc.unstaged_tiles < h_sfc.n_tiles // 2
    a, sa = ifl.if_filter(h_sfc, fields, ells, 1, solver=1, mg_min_ell=1.0)
    b, sb = ifl.if_filter(h_raw, fields, ells, 1, solver=1, mg_min_ell=1.0)
    jac, sj = ifl.if_filter(h_raw, fields, ells, 1)
    assert sa["code"] == 0 and sb["code"] == 0
    assert sb["iters"].sum() < sj["iters"].sum()          # the multigrid path did run
    a, b = a.cpu().numpy(), b.cpu().numpy()
    for f in range(fields.shape[0]):
        for j, ell in enumerate(ells):
            x, info = om.solve(fields[f], float(ell), 1)
            assert info["status"] == 0
            assert rel(a[f, j], x) <= TOL_FIELD and rel(b[f, j], x) <= TOL_FIELD, (f, j)
    h_sfc.close(); h_raw.close()


def test_multigrid_small_scales_through_the_hierarchy(ifl, oracle_mod):
    """Scales at and below the mean edge sent through the V cycle (mg_min_ell far below them): the systems are
    mass-dominated there, and the Galerkin mass matrices of the coarse levels are not diagonal -- the smoother's
    damping has to cover rho(D_M^-1 M_l) (2 to 3.6 on these hierarchies), or smooth error grows on the coarse
    levels.  The answers are the oracle's, in fewer iterations than Jacobi-PCG (28 673 vertices: four levels)."""
    w = make_config(4, level=6, n_ells=4)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period, flags=ifl.IF_FLAG_MULTIGRID)
    ells = h.mean_edge * np.array([0.5, 1.0, 2.0, 4.0])
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out, st = ifl.if_filter(h, w.fields, ells, 1, solver=1, mg_min_ell=0.1)
    jac, sj = ifl.if_filter(h, w.fields, ells, 1)
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["rel_res"] <= 1e-12)
    assert st["iters"].max() <= 40 and np.all(st["iters"][:, 1:] < sj["iters"][:, 1:])
    out = out.cpu().numpy()
    for f in range(w.fields.shape[0]):
        for j, ell in enumerate(ells):
            x, info = om.solve(w.fields[f], float(ell), 1)
            assert info["status"] == 0 and rel(out[f, j], x) <= TOL_FIELD, (f, j)
    h.close()


def test_multigrid_hierarchy_survives_save_and_load(ifl, tmp_path):
    """if_save / if_load of a handle prepared with IF_FLAG_MULTIGRID: the hierarchy is stored with the mesh, the loaded
    handle solves with solver = 1 (n = 1 and n = 2) and gives the same iteration counts and bits; a truncated or padded
    file is refused."""
    w = make_config(4, level=5, n_ells=7)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    a, sa = ifl.if_filter(h, w.fields, w.ells, 1, solver=1, mg_min_ell=2.0)
    path = str(tmp_path / "mesh_mg.bin")
    ifl.if_save(h, path)
    h2 = ifl.if_load(path)
    b, sb = ifl.if_filter(h2, w.fields, w.ells, 1, solver=1, mg_min_ell=2.0)
    assert np.array_equal(sa["iters"], sb["iters"]) and sa["iters"].max() < 60
    assert bool((a == b).all())
    i1, i2 = ifl.if_mesh_multigrid_info(h), ifl.if_mesh_multigrid_info(h2)
    assert i1["rows"] == i2["rows"] and i1["nnz"] == i2["nnz"] and i2["levels"] >= 3 and i2["build_seconds"] == 0.0
    c, sc = ifl.if_filter(h, w.fields, w.ells[:4], 2, solver=1)
    d, sd = ifl.if_filter(h2, w.fields, w.ells[:4], 2, solver=1)
    assert sc["mg_batch_iters"] > 0 and np.array_equal(sc["iters"], sd["iters"]) and bool((c == d).all())
    h.close(); h2.close()
    import os
    size = os.path.getsize(path)
    with open(path, "r+b") as fh:
        fh.truncate(size - 64)
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_load(path)
    assert e.value.code == -8
    with open(path, "ab") as fh:
        fh.write(b"\0" * 128)
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_load(path)
    assert e.value.code == -8


# ------------------------------------------------------------------------------------------ n = 2 at the top of its range
def true_residual(ifl, h, x, phi, area, ell, order_n):
    """||M phi - A_l x||_2 / ||M phi||_2 with A_l x from the library's if_apply (x: device tensor [V])."""
    import torch
    b = torch.from_numpy(area * phi).to(x.device)
    ax = ifl.if_apply(h, x[None, :], np.array([ell]), order_n)[0, 0]
    return float(torch.linalg.norm(b - ax) / torch.linalg.norm(b))


def parity_tolerance(area, phi, x_ref, res_a, res_b):
    """Tolerance for the relative L2 difference of two approximate solutions of A x = M phi, A = M + c S M^-1 S
    ("n = 2 at large scales"): x_a - x_b = A^-1 (r_b - r_a) and A >= M (S M^-1 S is positive
    semidefinite), so ||x_a - x_b|| <= (res_a + res_b) ||M phi|| / min A_v with res = TRUE relative residuals.
    1e-7 (north_star) wherever that bound supports it, the bound itself elsewhere."""
    bound = (res_a + res_b) * np.linalg.norm(area * phi) / area.min() / np.linalg.norm(x_ref)
    return max(TOL_FIELD, float(bound))


LARGE_N2 = {
    "cfg3_L4": lambda: make_config(3, level=4, n_ells=6, ell_max=32.0),
    "cfg3_L5": lambda: make_config(3, level=5, n_ells=6, ell_max=32.0),
    "cfg5_L5": lambda: make_config(5, level=5, n_fields=3, n_ells=6, ell_max=32.0),
}


@pytest.mark.parametrize("name", list(LARGE_N2))
def test_biharmonic_up_to_32_edge_lengths_matches_oracle(ifl, oracle_mod, name):
    """Reading A16 sets the n = 2 range to [1, 32] h; kappa ~ 1/2 (l^2 lambda_max)^2 reaches 1e8 at the top, where the
    true residual of any fp64 CG floors near u kappa (oracle: 1e-8 to 5e-8 at 32 h).  Scales 1, 2, 4, 8, 16, 32 h,
    every field element by element against the oracle, tolerance from the recorded true residuals of BOTH sides."""
    w = LARGE_N2[name]()
    assert abs(w.ells[-1] / w.mesh.h - 32.0) < 1e-9
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    area = om.area()
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    out, st = ifl.if_filter(h, w.fields, w.ells, 2)
    assert st["code"] == 0 and np.all(st["status"] == 0)
    sp = ifl.if_spectrum(h, w.fields, w.ells, 2)
    worst = 0.0
    for f in range(w.fields.shape[0]):
        en = []
        for j, ell in enumerate(w.ells):
            x, info = om.solve(w.fields[f], float(ell), 2)
            assert info["status"] == 0
            res_gpu = true_residual(ifl, h, out[f, j], w.fields[f], area, float(ell), 2)
            tol = parity_tolerance(area, w.fields[f], x, res_gpu, info["true_res"])
            err = rel(out[f, j].cpu().numpy(), x)
            assert err <= tol, (f, j, err, tol, res_gpu, info["true_res"])
            assert res_gpu <= 20.0 * max(info["true_res"], 1e-12), (f, j, res_gpu, info["true_res"])
            worst = max(worst, err)
            en.append(om.energy(x))
        en = np.array(en)
        k_mid, E = oracle_mod.spectrum(w.ells, en)
        assert np.all(np.abs(sp["energy"][f] - en) <= TOL_BIN * en)
        assert np.all(np.abs(sp["E"][f] - E) <= TOL_BIN * np.abs(E)), (f, np.abs(sp["E"][f] / E - 1).max())
    print(f"{name}: worst relative L2 difference from the oracle {worst:.2e}")
    h.close()


def test_biharmonic_32_edge_lengths_against_dense_direct_solve(ifl, oracle_mod):
    """The same top-of-range solves against numpy's dense LU of A = M + c S M^-1 S built from the oracle's CSR
    (2 562 vertices): neither CG is the reference here."""
    w = LARGE_N2["cfg3_L4"]()
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    rp, col, val = om.csr()
    V = om.nv
    S = np.zeros((V, V))
    for v in range(V):
        S[v, col[rp[v]:rp[v + 1]]] = val[rp[v]:rp[v + 1]]
    area = om.area()
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    ells = w.ells[-3:]
    out, st = ifl.if_filter(h, w.fields, ells, 2)
    assert st["code"] == 0
    for j, ell in enumerate(ells):
        A = np.diag(area) + 0.5 * ell ** 4 * (S @ (S / area[:, None]))
        x = np.linalg.solve(A, area * w.fields[0])
        assert rel(out[0, j].cpu().numpy(), x) <= TOL_FIELD, (j, rel(out[0, j].cpu().numpy(), x))
    h.close()


def test_biharmonic_beyond_its_range_returns_a_status(ifl):
    """for the biharmonic filter "the convergence can be lost for large l".  l = 400 h on a
    level-5 sphere (kappa ~ 1e12-1e13, far beyond reading A16's range): with a cap of 3 000 iterations the call must
    come back with status 1 for exactly those right-hand sides (finite output = the last iterate, the in-range column
    of the same batch converged); with the default cap it must come back as well, converged or not -- never hang."""
    w = make_config(5, level=5, n_fields=2, n_ells=2, ell_max=2.0)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    ells = w.mesh.h * np.array([2.0, 400.0])
    out, st = ifl.if_filter(h, w.fields, ells, 2, max_iter=3000)
    assert st["code"] == 1 and np.all(st["status"][:, 0] == 0) and np.all(st["status"][:, 1] == 1)
    assert np.all(st["iters"][:, 1] == 3000) and np.all(st["rel_res"][:, 1] > 1e-12)
    assert bool(out.isfinite().all())
    out, st = ifl.if_filter(h, w.fields, ells, 2)
    assert st["code"] in (0, 1) and np.all(np.isin(st["status"], (0, 1, 2)))
    assert st["code"] == (1 if np.any(st["status"] != 0) else 0) and st["iters"].max() <= 200000
    assert bool(out.isfinite().all())
    print("l = 400 h: status", st["status"][:, 1], "iterations", st["iters"][:, 1], "residual", st["rel_res"][:, 1])
    h.close()


def test_breakdown_status_is_per_column(ifl, oracle_mod):
    """status 2 (breakdown): a right-hand side whose arithmetic leaves the finite range stops with status 2 and does
    not disturb the other columns of its batch.  (a) a field holding a NaN; (b) l = 1e60 with n = 2: c = l^4 / 2
    overflows ||r0||^2."""
    w = make_config(4, level=4, n_fields=2, n_ells=3)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    fields = w.fields.copy()
    fields[1, 17] = np.nan
    out, st = ifl.if_filter(h, fields, w.ells, 1)
    assert st["code"] == 1 and np.all(st["status"][1] == 2) and np.all(st["status"][0] == 0)
    for j, ell in enumerate(w.ells):
        x, _ = om.solve(fields[0], float(ell), 1)
        assert rel(out[0, j].cpu().numpy(), x) <= TOL_FIELD
    ells = np.array([w.ells[0], 1e60])
    out, st = ifl.if_filter(h, w.fields, ells, 2)
    assert st["code"] == 1 and np.all(st["status"][:, 1] == 2) and np.all(st["status"][:, 0] == 0)
    for f in range(2):
        x, _ = om.solve(w.fields[f], float(ells[0]), 2)
        assert rel(out[f, 0].cpu().numpy(), x) <= TOL_FIELD
    h.close()


# ------------------------------------------------------------------------------------------ general unstructured meshes
@pytest.mark.parametrize("sell_c", [32, 64])
def test_rows_wider_than_eight_entries(ifl, oracle_mod, sell_c):
    """A Delaunay mesh with valences 3 to 14: SELL slices wider than the 8 slots the unrolled gather of the staged
    tiles handles.  Operator and solves (n = 1, 2, and the multigrid path, whose level 0 is the same kernel) against
    the oracle."""
    from workloads import delaunay_mesh
    m = delaunay_mesh(48, np.random.default_rng(3))
    om = oracle_mod.OracleMesh(m.coords, m.tri, None)
    rp, _, _ = om.csr()
    assert (np.diff(rp) - 1).max() >= 12
    rng = np.random.default_rng(4)
    fields = rng.standard_normal((3, m.n_vert))
    ells = np.array([0.8, 3.0, 9.0])
    h = ifl.if_prepare(m.coords, m.tri, None, sell_c=sell_c, flags=ifl.IF_FLAG_MULTIGRID)
    assert h.unstaged_tiles < h.n_tiles            # the wide rows sit in staged tiles
    for order_n in (1, 2):
        ap = ifl.if_apply(h, fields, ells, order_n).cpu().numpy()
        for f in range(3):
            for j, ell in enumerate(ells):
                assert rel(ap[f, j], om.apply(fields[f], float(ell), order_n)) <= 1e-12, (order_n, f, j)
    for order_n, kw in ((1, {}), (2, {}), (1, dict(solver=1, mg_min_ell=1.0))):
        out, st = ifl.if_filter(h, fields, ells[:2] if order_n == 2 else ells, order_n, **kw)
        assert st["code"] == 0
        out = out.cpu().numpy()
        for f in range(3):
            for j in range(out.shape[1]):
                x, info = om.solve(fields[f], float(ells[j]), order_n)
                assert info["status"] == 0 and rel(out[f, j], x) <= TOL_FIELD, (order_n, kw, f, j)
    h.close()


@pytest.mark.parametrize("check_every", [1, 3, 16])
def test_refill_while_other_columns_have_a_pending_step(ifl, oracle_mod, check_every):
    """4 columns, 27 short solves at a loose tolerance, graph launches of 1, 3 or 16 iterations: columns stop on odd and
    even iterations while the queue is not empty, so refilled columns restart next to columns whose last step
    x += alpha p is still pending.  At the same iteration count the CG iterate is the oracle's up to rounding."""
    from workloads import log_spaced
    # (mild jitter, no slivers: on config 2's literal mesh kappa amplifies the rounding of two CG implementations
    # to 1e-7 within a few hundred iterations, which would hide the defect this test is about)
    m = grid_mesh(48, periodic=True, jitter=0.2, random_diagonals=True, rng=np.random.default_rng(8))
    fields = np.random.default_rng(9).standard_normal((3, m.n_vert))
    ells = log_spaced(0.7, 4.0, 9)
    w = type("W", (), dict(mesh=m, fields=fields, ells=ells))
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    for order_n in (1, 2):
        out, st = ifl.if_filter(h, w.fields, w.ells, order_n, batch=4, tol=1e-4, check_every=check_every)
        out = out.cpu().numpy()
        assert st["code"] == 0
        same = 0
        for f in range(3):
            for j, ell in enumerate(w.ells):
                x, info = om.solve(w.fields[f], float(ell), order_n, tol=1e-4)
                if info["iters"] == st["iters"][f, j]:
                    same += 1
                    # n = 1: the two implementations agree to 1e-14 here; n = 2 (200-470 iterations on white noise)
                    # amplifies their rounding to 6e-7 with or without refill -- a misapplied last step is >= 1e-5
                    assert rel(out[f, j], x) <= (1e-12 if order_n == 1 else 5e-6), (order_n, f, j, rel(out[f, j], x))
                else:
                    # (n = 2: a few hundred iterations on white noise move the stop of two implementations by a few)
                    assert abs(info["iters"] - st["iters"][f, j]) <= (1 if order_n == 1 else 4) and rel(out[f, j], x) <= 1e-3
        assert same >= (24 if order_n == 1 else 14)
    h.close()


# ------------------------------------------------------------------------------------------ n = 2 through the hierarchy
@pytest.mark.parametrize("name", list(LARGE_N2))
def test_biharmonic_multigrid_product_preconditioner_matches_oracle(ifl, oracle_mod, name):
    """solver = 1 for n = 2: PCG on M + c S M^-1 S with B = V M V (V = one V cycle for M + sqrt(c) S).  Same systems,
    same start vector, same stop test as the oracle's Jacobi-PCG: fields at 1 ... 32 h within the tolerance derived
    from both true residuals, spectra to 1e-6, an order of magnitude fewer iterations at the large scales."""
    w = LARGE_N2[name]()
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    area = om.area()
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period, flags=ifl.IF_FLAG_MULTIGRID)
    out, st = ifl.if_filter(h, w.fields, w.ells, 2, solver=1, mg_min_ell=0.5)
    jac, stj = ifl.if_filter(h, w.fields, w.ells, 2)
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["rel_res"] <= 1e-12)
    print(name, "iterations multigrid", st["iters"][0], "Jacobi", stj["iters"][0])
    assert st["iters"].max() < 200 and st["iters"][:, -1].max() * 10 < stj["iters"][:, -1].min()
    sp = ifl.if_spectrum(h, w.fields, w.ells, 2, solver=1, mg_min_ell=0.5)
    worst = 0.0
    for f in range(w.fields.shape[0]):
        en = []
        for j, ell in enumerate(w.ells):
            x, info = om.solve(w.fields[f], float(ell), 2)
            assert info["status"] == 0
            res_gpu = true_residual(ifl, h, out[f, j], w.fields[f], area, float(ell), 2)
            tol = parity_tolerance(area, w.fields[f], x, res_gpu, info["true_res"])
            err = rel(out[f, j].cpu().numpy(), x)
            assert err <= tol, (f, j, err, tol, res_gpu, info["true_res"])
            worst = max(worst, err)
            en.append(om.energy(x))
        en = np.array(en)
        k_mid, E = oracle_mod.spectrum(w.ells, en)
        assert np.all(np.abs(sp["energy"][f] - en) <= TOL_BIN * en)
        assert np.all(np.abs(sp["E"][f] - E) <= TOL_BIN * np.abs(E))
    print(f"{name}: worst relative L2 difference from the oracle {worst:.2e}")
    h.close()


@pytest.mark.parametrize("turnover", ["host", "device"])
@pytest.mark.parametrize("order_n", [1, 2])
def test_multigrid_stream_refills_columns_and_is_deterministic(ifl, oracle_mod, order_n, turnover, monkeypatch):
    """More right-hand sides than columns (3 fields x 11 scales = 33 through 16 columns), very unequal scales: stopped
    columns are restarted from the queue at iteration boundaries next to running ones.  The preconditioner is a fixed
    operator per column, so two runs give the same iteration counts and the same bits; answers are the oracle's.
    Both ways of ending and starting columns: by the host one launch behind, and on the device inside the graph."""
    monkeypatch.setenv("IF_MG_HOST_REFILL", "1" if turnover == "host" else "0")
    w = make_config(5 if order_n == 2 else 4, level=5, n_fields=3, n_ells=11, ell_max=32.0)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    area = om.area()
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    a, sa = ifl.if_filter(h, w.fields, w.ells, order_n, solver=1, mg_min_ell=0.5)
    b, sb = ifl.if_filter(h, w.fields, w.ells, order_n, solver=1, mg_min_ell=0.5)
    assert sa["code"] == 0 and np.array_equal(sa["iters"], sb["iters"]) and bool((a == b).all())
    assert sa["mg_batch_iters"] > 0 and sa["mg_batch_iters"] == sa["batch_iters"]
    assert sa["iters"].sum() <= 16 * sa["mg_batch_iters"]
    for f in range(3):
        for j in (0, 3, 5, 8, 10):
            x, info = om.solve(w.fields[f], float(w.ells[j]), order_n)
            res_gpu = true_residual(ifl, h, a[f, j], w.fields[f], area, float(w.ells[j]), order_n)
            tol = parity_tolerance(area, w.fields[f], x, res_gpu, info["true_res"])
            assert info["status"] == 0 and rel(a[f, j].cpu().numpy(), x) <= tol, (f, j)
    # mixed: the smallest scales stay on the Jacobi path, and the iteration cap gives a status in the multigrid path
    c, sc = ifl.if_filter(h, w.fields, w.ells, order_n, solver=1, mg_min_ell=3.0)
    assert sc["code"] == 0 and 0 < sc["mg_batch_iters"] < sc["batch_iters"]
    assert float((c - a).abs().max()) <= 1e-8 * float(a.abs().max())
    d, sd = ifl.if_filter(h, w.fields[:1], w.ells[-1:], order_n, solver=1, max_iter=3)
    assert sd["code"] == 1 and sd["status"][0, 0] == 1 and sd["iters"][0, 0] == 3 and bool(d.isfinite().all())
    h.close()


@pytest.mark.parametrize("order_n", [1, 2])
def test_multigrid_turnover_on_device_matches_host_refill(ifl, oracle_mod, order_n, monkeypatch, capfd):
    """The multigrid stream ends and starts its columns on the device (k_turn_plan inside every iteration's graph;
    the host only watches).  Against the host-driven refill of the Jacobi path's loop (IF_MG_HOST_REFILL=1), which
    sees a stop one launch late: the same per-right-hand-side arithmetic, so the same iteration counts and fields to
    rounding, in fewer fused iterations; for fewer right-hand sides than columns, exactly 16, and many more; filter,
    high-pass and spectrum jobs; answers are the oracle's."""
    w = make_config(5 if order_n == 2 else 4, level=5, n_fields=5, n_ells=9, ell_max=24.0)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    area = om.area()
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    for nf, ne in ((1, 3), (2, 8), (5, 9)):                      # 3, 16 and 45 right-hand sides
        fields, ells = w.fields[:nf], w.ells[:ne]
        monkeypatch.setenv("IF_MG_HOST_REFILL", "0")             # (unset: by mesh size, the host on a mesh this small)
        monkeypatch.setenv("IF_VERBOSE", "1")
        capfd.readouterr()
        dev, sd = ifl.if_filter(h, fields, ells, order_n, solver=1, mg_min_ell=0.5)
        trace = capfd.readouterr().err
        monkeypatch.delenv("IF_VERBOSE")
        if nf * ne > 8:      # the tail of the stream really moves to the narrower kernels (16 -> 8 or 4, 8 -> 4)
            assert "tail moved from 16 to" in trace, trace
        spd = ifl.if_spectrum(h, fields, ells, order_n, solver=1, mg_min_ell=0.5)
        monkeypatch.setenv("IF_MG_HOST_REFILL", "1")
        host, sh = ifl.if_filter(h, fields, ells, order_n, solver=1, mg_min_ell=0.5)
        sph = ifl.if_spectrum(h, fields, ells, order_n, solver=1, mg_min_ell=0.5)
        monkeypatch.delenv("IF_MG_HOST_REFILL")
        assert sd["code"] == 0 and sh["code"] == 0 and spd["stats"]["code"] == 0
        assert sd["mg_batch_iters"] == sd["batch_iters"] > 0
        assert np.array_equal(sd["status"], sh["status"])
        assert np.abs(sd["iters"].astype(np.int64) - sh["iters"]).max() <= 1, (sd["iters"], sh["iters"])
        assert sd["mg_batch_iters"] <= sh["mg_batch_iters"], (nf, ne, sd["mg_batch_iters"], sh["mg_batch_iters"])
        if nf * ne > 16:
            assert sd["mg_batch_iters"] < sh["mg_batch_iters"]           # the refills no longer idle an iteration
        scale = float(host.abs().max())
        assert float((dev - host).abs().max()) <= 1e-9 * scale
        assert np.all(np.abs(spd["energy"] - sph["energy"]) <= 1e-9 * sph["energy"])
        d = dev.cpu().numpy()
        en = 0.5 * (area * d * d).sum(axis=-1) / area.sum()             # the plain definition on the returned fields
        assert np.all(np.abs(spd["energy"] - en) <= 1e-9 * en)
    # the oracle, on a sample of the largest case
    for f, j in ((0, 0), (2, 4), (4, 8), (3, 6)):
        x, info = om.solve(w.fields[f], float(w.ells[j]), order_n)
        res_gpu = true_residual(ifl, h, dev[f, j], w.fields[f], area, float(w.ells[j]), order_n)
        tol = parity_tolerance(area, w.fields[f], x, res_gpu, info["true_res"])
        assert info["status"] == 0 and rel(dev[f, j].cpu().numpy(), x) <= tol, (f, j)
    # high-pass output and the iteration cap through the device turnover
    monkeypatch.setenv("IF_MG_HOST_REFILL", "0")
    hp, shp = ifl.if_filter(h, w.fields[:3], w.ells, order_n, solver=1, mg_min_ell=0.5, flags=ifl.IF_FLAG_HIGHPASS)
    import torch
    phi = torch.from_numpy(w.fields[:3]).to(hp.device)[:, None, :]
    assert float((hp - (phi - dev[:3])).abs().max()) <= 1e-9 * scale
    cap, sc = ifl.if_filter(h, w.fields, w.ells, order_n, solver=1, mg_min_ell=0.5, max_iter=4)
    assert sc["code"] == 1 and int(sc["iters"].max()) == 4 and bool(cap.isfinite().all())
    assert np.all(((sc["status"] == 0) & (sc["iters"] <= 4)) | ((sc["status"] == 1) & (sc["iters"] == 4)))
    h.close()


def test_default_split_between_the_paths_depends_on_the_number_of_columns(ifl):
    """mg_min_ell = 0 (default): with 12 or more right-hand sides every scale from 0.5 mean edges goes through the
    multigrid stream; a call with fewer runs the 4- or 8-column variants of the cycle's kernels, which cost more per
    right-hand side, so its smallest scales stay on Jacobi-PCG up to the measured break-even (2.5 edge lengths for up
    to 4 columns, 1.5 for up to 11, n = 1; 1 for n = 2).  The answers do not depend on the split nor on the width."""
    w = make_config(4, level=5, n_fields=2, n_ells=8, ell_max=32.0)        # scales 1, 1.6, 2.7, 4.4, 7.2, 12, 20, 32 h
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    scale = None
    for order_n, top in ((1, 8), (2, 6)):
        ells = w.ells[:top]
        ref, sr = ifl.if_filter(h, w.fields, ells, order_n)                    # Jacobi-PCG
        scale = float(ref.abs().max())
        many, sm = ifl.if_filter(h, w.fields, ells, order_n, solver=1)         # 12-16 right-hand sides: all in the stream
        assert sm["code"] == 0 and sm["mg_batch_iters"] == sm["batch_iters"] > 0
        few_small, s1 = ifl.if_filter(h, w.fields[:1], ells[:1], order_n, solver=1)          # one, just below one mean edge
        assert s1["code"] == 0 and s1["mg_batch_iters"] == 0
        forced, s2 = ifl.if_filter(h, w.fields[:1], ells[:3], order_n, solver=1, mg_min_ell=0.5)     # 4 columns
        assert s2["mg_batch_iters"] == s2["batch_iters"] > 0
        few_large, s3 = ifl.if_filter(h, w.fields[:1], ells[3:6], order_n, solver=1)         # 3 beyond 2.5 edges
        assert s3["mg_batch_iters"] == s3["batch_iters"] > 0
        mixed, s4 = ifl.if_filter(h, w.fields[:1], ells, order_n, solver=1)    # 6-8 right-hand sides: 8 columns
        assert (0 < s4["mg_batch_iters"] < s4["batch_iters"]) if order_n == 1 else s4["mg_batch_iters"] > 0
        tol = (1e-9 if order_n == 1 else 1e-7) * scale
        for got, want in ((many, ref), (few_small, ref[:1, :1]), (forced, ref[:1, :3]), (few_large, ref[:1, 3:6]),
                          (mixed, ref[:1])):
            assert float((got - want).abs().max()) <= tol, order_n
    h.close()


def test_legacy_default_stream_runs_without_graphs(ifl, monkeypatch):
    """Stream 0 (the legacy default stream) cannot be captured: both stream loops then launch their kernels directly.
    Same kernels in the same order, so the same bits as the graph path on a side stream -- Jacobi-PCG, the multigrid
    stream with the host-driven refill and with the turnover on the device."""
    import torch
    w = make_config(4, level=5, n_fields=3, n_ells=7, ell_max=24.0)                # 21 right-hand sides
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    legacy = torch.cuda.default_stream()
    assert legacy.cuda_stream == 0
    for opts, env in ((dict(), None), (dict(solver=1, mg_min_ell=0.5), "1"), (dict(solver=1, mg_min_ell=0.5), "0")):
        if env is None:
            monkeypatch.delenv("IF_MG_HOST_REFILL", raising=False)
        else:
            monkeypatch.setenv("IF_MG_HOST_REFILL", env)
        a, sa = ifl.if_filter(h, w.fields, w.ells, 1, **opts)                      # the binding's side stream: graphs
        b, sb = ifl.if_filter(h, w.fields, w.ells, 1, stream=legacy, **opts)       # stream 0: direct launches
        assert sa["code"] == 0 and sb["code"] == 0
        assert np.array_equal(sa["iters"], sb["iters"]) and bool((a == b).all()), (opts, env)
        assert sa["batch_iters"] == sb["batch_iters"]
        spa = ifl.if_spectrum(h, w.fields, w.ells, 1, **opts)
        spb = ifl.if_spectrum(h, w.fields, w.ells, 1, stream=legacy, **opts)
        assert np.array_equal(spa["energy"], spb["energy"]) and np.array_equal(spa["E"], spb["E"])
    h.close()


# ------------------------------------------------------------------------------------------ higher orders, velocity pairs
@pytest.mark.parametrize("order_n", [3, 4])
def test_higher_order_filters_match_oracle(ifl, oracle_mod, order_n):
    """n = 3, 4 ("can be generalized to higher-order filters"; PAPER.md:201-205 uses the four-Laplacian
    filter): operator (1e-12), config 1 against the closed form 1 / (1 + gamma (l^2 lambda)^n), a level-4 sphere against
    the oracle with the tolerance derived from both true residuals (A >= M for every order), spectra to 1e-6, all three
    column widths with a ragged tail.  Scales stay where fp64 carries the order: kappa ~ 1/2 (l^2 lambda_max)^n."""
    top = 4.0 if order_n == 3 else 2.2
    w1 = make_config(1, n_ells=5, ell_max=top)
    N = 64
    wv = w1.waves[0]
    lam = 4.0 - 2.0 * np.cos(2 * np.pi * wv.k[:, 0] / N) - 2.0 * np.cos(2 * np.pi * wv.k[:, 1] / N)
    basis = np.cos(w1.mesh.coords @ (wv.k.T * wv.scale) + wv.theta)
    h = ifl.if_prepare(w1.mesh.coords, w1.mesh.tri, w1.mesh.period)
    out, st = ifl.if_filter(h, w1.fields, w1.ells, order_n)
    assert st["code"] == 0
    for j, ell in enumerate(w1.ells):
        ref = basis @ (wv.amp / (1.0 + 0.5 * (ell ** 2 * lam) ** order_n))
        assert rel(out[0, j].cpu().numpy(), ref) <= TOL_FIELD, j
    h.close()
    w = make_config(3, level=4, n_fields=3, n_ells=5, ell_max=top)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    area = om.area()
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID)
    ap = ifl.if_apply(h, w.fields, w.ells, order_n).cpu().numpy()
    for f in range(3):
        for j, ell in enumerate(w.ells):
            assert rel(ap[f, j], om.apply(w.fields[f], float(ell), order_n)) <= 1e-12, (f, j)
    ref = {}
    for batch in (16, 8, 4):
        out, st = ifl.if_filter(h, w.fields, w.ells, order_n, batch=batch, solver=1)   # (multigrid does not serve n > 2)
        assert st["code"] == 0 and st["mg_batch_iters"] == 0
        for f in range(3):
            for j, ell in enumerate(w.ells):
                if (f, j) not in ref:
                    ref[f, j] = om.solve(w.fields[f], float(ell), order_n)
                x, info = ref[f, j]
                assert info["status"] == 0
                res_gpu = true_residual(ifl, h, out[f, j], w.fields[f], area, float(ell), order_n)
                tol = parity_tolerance(area, w.fields[f], x, res_gpu, info["true_res"])
                assert rel(out[f, j].cpu().numpy(), x) <= tol, (batch, f, j, tol)
                # the same exact Jacobi diagonal as the oracle's: the library (tol 1e-12) stops a little before the
                # oracle (1e-13), never later, and not by much
                assert 0.7 * info["iters"] <= int(st["iters"][f, j]) <= info["iters"] + 3
    sp = ifl.if_spectrum(h, w.fields, w.ells, order_n)
    for f in range(3):
        en = np.array([om.energy(ref[f, j][0]) for j in range(len(w.ells))])
        k_mid, E = oracle_mod.spectrum(w.ells, en)
        assert np.all(np.abs(sp["energy"][f] - en) <= TOL_BIN * en) and np.all(np.abs(sp["E"][f] - E) <= TOL_BIN * np.abs(E))
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h, w.fields, w.ells, 5)
    assert e.value.code == -1
    h.close()


def test_velocity_pairs_spectrum(ifl, oracle_mod):
    """IF_FLAG_PAIRS: fields are (u, v) pairs and the two per-field spectra are added (reading A4: "for (u, v) the caller
    adds the two per-field spectra"; the kinetic-energy spectra of PAPER.md:149-157)."""
    w = make_config(5, level=4, n_fields=4, n_ells=5, ell_max=6.0)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None)
    for order_n in (1, 2):
        en = np.array([[om.energy(om.solve(w.fields[f], float(l), order_n)[0]) for l in w.ells] for f in range(4)])
        sp = ifl.if_spectrum(h, w.fields, w.ells, order_n, flags=ifl.IF_FLAG_PAIRS)
        single = ifl.if_spectrum(h, w.fields, w.ells, order_n)
        assert sp["energy"].shape == (2, 5) and sp["E"].shape == (2, 4) and sp["stats"]["iters"].shape == (4, 5)
        for p in range(2):
            ke = en[2 * p] + en[2 * p + 1]
            k_mid, E = oracle_mod.spectrum(w.ells, ke)
            assert np.all(np.abs(sp["energy"][p] - ke) <= TOL_BIN * ke)
            assert np.all(np.abs(sp["E"][p] - E) <= TOL_BIN * np.abs(E))
            assert np.allclose(sp["E"][p], single["E"][2 * p] + single["E"][2 * p + 1], rtol=1e-12)
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_spectrum(h, w.fields[:3], w.ells, 1, flags=ifl.IF_FLAG_PAIRS)
    assert e.value.code == -1
    h.close()


# ------------------------------------------------------------------------------------------ vector filter with metric terms
def vector_workload(level, n_pairs, seed=21):
    from workloads import icosphere, jitter_sphere, sphere_band, sphere_velocity_field
    mesh = sphere_band(jitter_sphere(icosphere(level), 0.2, np.random.default_rng(seed)), 70.0)
    rng = np.random.default_rng(seed + 1)
    fields = np.empty((2 * n_pairs, mesh.n_vert))
    for p in range(n_pairs):
        fields[2 * p], fields[2 * p + 1] = sphere_velocity_field(mesh.coords, 3 * 2 ** (level - 3), 24, rng)
    return mesh, fields


@pytest.mark.parametrize("order_n", [1, 2])
def test_vector_filter_matches_oracle(ifl, oracle_mod, order_n):
    """IF_FLAG_VECTOR: (u, v) pairs filtered as coupled 2V x 2V systems with the metric terms D~, T.
    Operator to 1e-12, coarse-grained velocities against the oracle's joint PCG with the tolerance derived from both
    true residuals (S_2 >= M_2: D_2 is positive semidefinite), kinetic-energy spectra (IF_FLAG_PAIRS) to 1e-6; three
    column widths, more pairs than columns (refill in pairs), and the scalar path of the same handle unchanged."""
    mesh, fields = vector_workload(5, 3)
    top = 20.0 if order_n == 1 else 8.0
    from workloads import log_spaced
    ells = mesh.h * log_spaced(1.0, top, 5)
    om = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    om.build_vector(1.0)
    area = om.area()
    VEC = ifl.IF_FLAG_VECTOR
    h = ifl.if_prepare(mesh.coords, mesh.tri, None, flags=VEC, radius=1.0)
    ap = ifl.if_apply(h, fields, ells, order_n, flags=VEC).cpu().numpy()
    ref = {}
    for p in range(3):
        for j, ell in enumerate(ells):
            ou, ov = om.apply_vector(fields[2 * p], fields[2 * p + 1], float(ell), order_n)
            assert rel(ap[2 * p, j], ou) <= 1e-12 and rel(ap[2 * p + 1, j], ov) <= 1e-12, (p, j)
            ref[p, j] = om.solve_vector(fields[2 * p], fields[2 * p + 1], float(ell), order_n)
            assert ref[p, j][2]["status"] == 0
    import torch
    for batch in (16, 8, 4):
        out, st = ifl.if_filter(h, fields, ells, order_n, flags=VEC, batch=batch)
        assert st["code"] == 0
        for p in range(3):
            bnorm = np.linalg.norm(np.concatenate([area * fields[2 * p], area * fields[2 * p + 1]]))
            for j, ell in enumerate(ells):
                xu, xv, info = ref[p, j]
                x = out[2 * p:2 * p + 2, j]
                ax = ifl.if_apply(h, x, np.array([ell]), order_n, flags=VEC)[:, 0].cpu().numpy()
                res_gpu = np.linalg.norm(np.concatenate([area * fields[2 * p] - ax[0], area * fields[2 * p + 1] - ax[1]])) / bnorm
                xr = np.concatenate([xu, xv])
                tol = max(TOL_FIELD, (res_gpu + info["true_res"]) * bnorm / area.min() / np.linalg.norm(xr))
                err = rel(np.concatenate([x[0].cpu().numpy(), x[1].cpu().numpy()]), xr)
                assert err <= tol, (batch, p, j, err, tol)
                assert st["iters"][2 * p, j] == st["iters"][2 * p + 1, j] and st["status"][2 * p, j] == 0
                assert 0.7 * info["iters"] <= st["iters"][2 * p, j] <= info["iters"] + 3
    sp = ifl.if_spectrum(h, fields, ells, order_n, flags=VEC | ifl.IF_FLAG_PAIRS)
    assert sp["energy"].shape == (3, 5)
    for p in range(3):
        ke = np.array([om.energy(ref[p, j][0]) + om.energy(ref[p, j][1]) for j in range(5)])
        k_mid, E = oracle_mod.spectrum(ells, ke)
        assert np.all(np.abs(sp["energy"][p] - ke) <= TOL_BIN * ke) and np.all(np.abs(sp["E"][p] - E) <= TOL_BIN * np.abs(E))
    # without the per-call flag the same handle filters scalars, and the coupling is not a small effect
    sc, _ = ifl.if_filter(h, fields[:2], ells[-1:], order_n)
    su, _ = om.solve(fields[0], float(ells[-1]), order_n)
    assert rel(sc[0, 0].cpu().numpy(), su) <= TOL_FIELD and rel(su, ref[0, 4][0]) > 1e-3
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h, fields[:3], ells, order_n, flags=VEC)               # odd number of fields
    assert e.value.code == -1
    h0 = ifl.if_prepare(mesh.coords, mesh.tri, None)
    with pytest.raises(ifl.ImplicitFilterError) as e:
        ifl.if_filter(h0, fields[:2], ells, order_n, flags=VEC)              # handle without metric terms
    assert e.value.code == -1
    h.close(); h0.close()


@pytest.mark.parametrize("turnover", ["host", "device"])
def test_vector_filter_through_the_multigrid_path(ifl, oracle_mod, turnover, monkeypatch, tmp_path):
    """solver = 1 with IF_FLAG_VECTOR (n = 1): PCG on the coupled 2V system preconditioned by the V cycle of the
    scalar hierarchy -- smoothing and residuals on the mesh with the coupled operator (metric terms D~, T), coarse
    correction per component.  Same systems, same start, same stop test: the oracle's joint PCG is the reference, with
    the tolerance derived from both true residuals; both columns of a pair share the iteration count; more pairs
    than columns (refill in pairs); far fewer iterations than Jacobi-PCG at the large scales; spectra of pairs."""
    monkeypatch.setenv("IF_MG_HOST_REFILL", "1" if turnover == "host" else "0")     # pairs end and start together
    mesh, fields = vector_workload(5, 10)                       # 10 (u, v) pairs = 20 fields
    from workloads import log_spaced
    ells = mesh.h * log_spaced(1.0, 48.0, 4)                    # 40 pair solves through 8 pair slots
    om = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    om.build_vector(1.0)
    area = om.area()
    VEC = ifl.IF_FLAG_VECTOR
    h = ifl.if_prepare(mesh.coords, mesh.tri, None, flags=VEC | ifl.IF_FLAG_MULTIGRID, radius=1.0)
    out, st = ifl.if_filter(h, fields, ells, 1, flags=VEC, solver=1, mg_min_ell=0.5)
    jac, sj = ifl.if_filter(h, fields, ells, 1, flags=VEC)
    assert st["code"] == 0 and sj["code"] == 0
    assert st["mg_batch_iters"] == st["batch_iters"] > 0 and sj["mg_batch_iters"] == 0
    assert np.array_equal(st["iters"][0::2], st["iters"][1::2])                 # a pair is one system
    assert int(st["iters"][:, -1].max()) * 4 < int(sj["iters"][:, -1].min())     # the large scale: far fewer iterations
    assert float((out - jac).abs().max()) <= 1e-8 * float(jac.abs().max())
    for p in (0, 4, 9):
        bnorm = np.linalg.norm(np.concatenate([area * fields[2 * p], area * fields[2 * p + 1]]))
        for j, ell in enumerate(ells):
            xu, xv, info = om.solve_vector(fields[2 * p], fields[2 * p + 1], float(ell), 1)
            assert info["status"] == 0
            x = out[2 * p:2 * p + 2, j]
            ax = ifl.if_apply(h, x, np.array([ell]), 1, flags=VEC)[:, 0].cpu().numpy()
            res_gpu = np.linalg.norm(np.concatenate([area * fields[2 * p] - ax[0], area * fields[2 * p + 1] - ax[1]])) / bnorm
            xr = np.concatenate([xu, xv])
            tol = max(TOL_FIELD, (res_gpu + info["true_res"]) * bnorm / area.min() / np.linalg.norm(xr))
            err = rel(np.concatenate([x[0].cpu().numpy(), x[1].cpu().numpy()]), xr)
            assert err <= tol and res_gpu <= 1e-10, (p, j, err, tol, res_gpu)
    sp = ifl.if_spectrum(h, fields, ells, 1, flags=VEC | ifl.IF_FLAG_PAIRS, solver=1, mg_min_ell=0.5)
    sq = ifl.if_spectrum(h, fields, ells, 1, flags=VEC | ifl.IF_FLAG_PAIRS)
    assert sp["energy"].shape == (10, 4) and np.all(np.abs(sp["energy"] - sq["energy"]) <= 1e-9 * sq["energy"])
    assert np.all(np.abs(sp["E"] - sq["E"]) <= TOL_BIN * np.abs(sq["E"]))
    # two runs: the same bits (a fixed operator per column), and n = 2 pairs stay on the Jacobi path
    again, _ = ifl.if_filter(h, fields, ells, 1, flags=VEC, solver=1, mg_min_ell=0.5)
    assert bool((again == out).all())
    # a handle with both the metric terms and the hierarchy through if_save / if_load: the same bits
    path = str(tmp_path / "vec_mg.ifm")
    ifl.if_save(h, path)
    h2 = ifl.if_load(path)
    loaded, sl = ifl.if_filter(h2, fields, ells, 1, flags=VEC, solver=1, mg_min_ell=0.5)
    assert sl["code"] == 0 and sl["mg_batch_iters"] == st["mg_batch_iters"] and bool((loaded == out).all())
    h2.close()
    # n = 2 pairs: the product preconditioner V M_2 V with the same coupled cycle (scales to 16 edge lengths)
    ells2 = mesh.h * log_spaced(1.0, 16.0, 4)
    b2, s2 = ifl.if_filter(h, fields[:6], ells2, 2, flags=VEC, solver=1, mg_min_ell=0.5)
    j2, sj2 = ifl.if_filter(h, fields[:6], ells2, 2, flags=VEC)
    assert s2["code"] == 0 and sj2["code"] == 0 and s2["mg_batch_iters"] == s2["batch_iters"] > 0
    assert np.array_equal(s2["iters"][0::2], s2["iters"][1::2])
    assert int(s2["iters"][:, -1].max()) * 10 < int(sj2["iters"][:, -1].min())
    for p in range(3):
        bnorm = np.linalg.norm(np.concatenate([area * fields[2 * p], area * fields[2 * p + 1]]))
        for j, ell in enumerate(ells2):
            res = []
            for x in (b2[2 * p:2 * p + 2, j], j2[2 * p:2 * p + 2, j]):
                ax = ifl.if_apply(h, x, np.array([ell]), 2, flags=VEC)[:, 0].cpu().numpy()
                res.append(np.linalg.norm(np.concatenate([area * fields[2 * p] - ax[0], area * fields[2 * p + 1] - ax[1]])) / bnorm)
            xa = np.concatenate([b2[2 * p, j].cpu().numpy(), b2[2 * p + 1, j].cpu().numpy()])
            xb = np.concatenate([j2[2 * p, j].cpu().numpy(), j2[2 * p + 1, j].cpu().numpy()])
            tol = max(TOL_FIELD, (res[0] + res[1]) * bnorm / area.min() / np.linalg.norm(xb))      # S_2 >= M_2
            assert rel(xa, xb) <= tol, (p, j, rel(xa, xb), tol, res)
            if p == 0 and j == 0:        # one pair or two alone: the 4- and 8-column variants of the coupled cycle
                for npairs in (1, 2):
                    for order_k in (1, 2):
                        want = (jac if order_k == 1 else j2)[:2 * npairs, 1:3]
                        ee = (ells if order_k == 1 else ells2)[1:3]
                        few, sf = ifl.if_filter(h, fields[:2 * npairs], ee, order_k, flags=VEC, solver=1, mg_min_ell=0.5)
                        assert sf["code"] == 0 and sf["mg_batch_iters"] == sf["batch_iters"] > 0
                        assert float((few - want).abs().max()) <= (1e-8 if order_k == 1 else 1e-6) * float(want.abs().max())
            if p == 0 and j <= 1:        # and the oracle's joint PCG where it finishes in seconds
                xu, xv, info = om.solve_vector(fields[0], fields[1], float(ell), 2)
                xr = np.concatenate([xu, xv])
                tol = max(TOL_FIELD, (res[0] + info["true_res"]) * bnorm / area.min() / np.linalg.norm(xr))
                assert info["status"] == 0 and rel(xa, xr) <= tol, (j, rel(xa, xr), tol)
    h.close()


def test_vector_filter_planar_mesh_and_save_load(ifl, oracle_mod, tmp_path):
    """A planar mesh has no metric terms: the vector filter returns the two scalar filters.  The metric arrays go
    through if_save / if_load."""
    m = grid_mesh(40, periodic=True, jitter=0.2, random_diagonals=True, rng=np.random.default_rng(31))
    fields = np.random.default_rng(32).standard_normal((2, m.n_vert))
    ells = np.array([0.8, 2.5, 6.0])
    h = ifl.if_prepare(m.coords, m.tri, m.period, flags=ifl.IF_FLAG_VECTOR)
    a, sa = ifl.if_filter(h, fields, ells, 1, flags=ifl.IF_FLAG_VECTOR)
    b, sb = ifl.if_filter(h, fields, ells, 1)
    assert sa["code"] == 0 and float((a - b).abs().max()) <= 1e-9 * float(b.abs().max())
    h.close()
    mesh, vf = vector_workload(4, 1)
    h = ifl.if_prepare(mesh.coords, mesh.tri, None, flags=ifl.IF_FLAG_VECTOR)     # radius 0 => mean |x_v| = 1
    c, sc = ifl.if_filter(h, vf, mesh.h * ells, 2, flags=ifl.IF_FLAG_VECTOR)
    path = str(tmp_path / "vec.ifm")
    ifl.if_save(h, path)
    h.close()
    g = ifl.if_load(path)
    d, sd = ifl.if_filter(g, vf, mesh.h * ells, 2, flags=ifl.IF_FLAG_VECTOR)
    assert sc["code"] == 0 and np.array_equal(sc["iters"], sd["iters"]) and bool((c == d).all())
    om = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    om.build_vector()
    xu, xv, info = om.solve_vector(vf[0], vf[1], float(mesh.h * ells[1]), 2)
    assert rel(c[0, 1].cpu().numpy(), xu) <= TOL_FIELD and rel(c[1, 1].cpu().numpy(), xv) <= TOL_FIELD
    g.close()


def test_true_residual_in_stats(ifl, oracle_mod):
    """IF_FLAG_TRUE_RESIDUAL: if_filter also reports ||M phi - A_l x|| / ||M phi|| of the fields it returns (SURVEY.md
    section 5 metrics).  Checked against the same quantity formed from if_apply in the test and against the oracle's
    recorded true residual (same floor u * kappa, within a factor); n = 1, 2, both solvers, narrow batches, the vector
    filter."""
    w = make_config(5, level=5, n_fields=3, n_ells=5, ell_max=32.0)
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    area = om.area()
    TR = ifl.IF_FLAG_TRUE_RESIDUAL
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_MULTIGRID | ifl.IF_FLAG_VECTOR)
    for order_n, kw in ((1, {}), (2, {}), (2, dict(solver=1)), (1, dict(batch=4))):
        out, st = ifl.if_filter(h, w.fields, w.ells, order_n, flags=TR, **kw)
        assert st["code"] == 0 and np.all(np.isfinite(st["true_res"]))
        for f in range(3):
            for j, ell in enumerate(w.ells):
                mine = true_residual(ifl, h, out[f, j], w.fields[f], area, float(ell), order_n)
                assert abs(st["true_res"][f, j] - mine) <= 1e-6 * mine + 1e-16, (order_n, kw, f, j)
                assert st["true_res"][f, j] >= 0.3 * st["rel_res"][f, j] - 1e-15
        _, info = om.solve(w.fields[0], float(w.ells[-1]), order_n)
        assert st["true_res"][0, -1] <= 20.0 * max(info["true_res"], 1e-12)
    _, st = ifl.if_filter(h, w.fields, w.ells, 1)
    assert np.all(np.isnan(st["true_res"]))                      # off by default
    out, st = ifl.if_filter(h, w.fields[:2], w.ells[:3], 1, flags=TR | ifl.IF_FLAG_VECTOR)
    assert st["code"] == 0 and np.array_equal(st["true_res"][0], st["true_res"][1]) and np.all(st["true_res"] <= 1e-11)
    h.close()
