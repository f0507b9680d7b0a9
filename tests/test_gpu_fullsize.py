"""Full-size checks on BASELINE.json config 4 in the launch configuration bench.py times (K = 16 columns, refill,
default tolerance): sampled right-hand sides against the oracle where it finishes in seconds, and properties that
hold at any size where it does not.  Needs a B200-class GPU (about 6 GB) and a few minutes."""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu

TOL_FIELD = 1e-7
TOL_BIN = 1e-6


@pytest.fixture(scope="module")
def full():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    if torch.cuda.get_device_properties(0).total_memory < 16e9:
        pytest.skip("needs 16 GB of device memory")
    import paper_2404_07398_b200 as lib
    lib.load_library()
    w = make_config(4)
    # as bench.py prepares it: with the multigrid hierarchy, which the default (Jacobi) solver does not touch
    h = lib.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period, flags=lib.IF_FLAG_MULTIGRID)
    yield lib, w, h
    h.close()


@pytest.fixture(scope="module")
def jacobi_spectrum(full):
    lib, w, h = full
    return lib.if_spectrum(h, w.fields, w.ells, 1)


@pytest.fixture(scope="module")
def oracle_mesh(full, oracle_mod):
    _, w, _ = full
    return oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_full_mesh_is_the_named_workload(full):
    lib, w, h = full
    assert w.mesh.n_vert == 7340033 and w.mesh.n_tri == 14664875      # 10 485 762 vertices minus the land mask
    assert h.n_vert == w.mesh.n_vert and w.n_rhs == 80 and w.order_n == 1
    assert abs(w.ells[-1] / w.mesh.h - 1000.0) < 1e-9 and abs(w.ells[0] / w.mesh.h - 1.0) < 1e-12
    # the tiled SpMM stages (nearly) every tile in shared memory on the space-filling-curve order
    assert h.n_tiles == (h.n_vert + 127) // 128 and h.unstaged_tiles <= 0.05 * h.n_tiles


def test_spectrum_full_size_properties_and_sampled_energies(full, oracle_mesh, jacobi_spectrum):
    """The bench step itself: all 80 right-hand sides.  e_l monotone, E >= 0, every solve converged; the energies of
    sampled right-hand sides (those the oracle finishes in seconds) to 1e-6."""
    lib, w, h = full
    sp = jacobi_spectrum
    st = sp["stats"]
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["rel_res"] <= 1e-12)
    assert np.all(np.diff(sp["energy"], axis=1) < 0.0)                  # strictly decreasing in l
    assert np.all(sp["E"] > 0.0)
    k = 1.0 / w.ells
    assert np.allclose(sp["k_mid"], np.sqrt(k[:-1] * k[1:]), rtol=1e-14)
    for f in range(2):                                                   # telescoping sum of the bins
        tele = np.sum(sp["E"][f] * (k[:-1] - k[1:]))
        assert abs(tele - (sp["energy"][f, 0] - sp["energy"][f, -1])) <= 1e-12 * sp["energy"][f, 0]
    for f, j in ((0, 0), (0, 8), (1, 4), (0, 16)):
        x, info = oracle_mesh.solve(w.fields[f], float(w.ells[j]), 1)
        assert info["status"] == 0
        e = oracle_mesh.energy(x)
        assert abs(sp["energy"][f, j] - e) <= TOL_BIN * e, (f, j)


def test_filter_full_size_sampled_fields(full, oracle_mesh):
    """16 right-hand sides (2 fields x the 8 smallest scales) in one K = 16 batch; three of them against the oracle."""
    lib, w, h = full
    ells = w.ells[:8]
    out, st = lib.if_filter(h, w.fields, ells, 1)
    assert st["code"] == 0
    for f, j in ((0, 0), (1, 3), (0, 7)):
        x, info = oracle_mesh.solve(w.fields[f], float(ells[j]), 1)
        assert info["status"] == 0
        assert rel(out[f, j].cpu().numpy(), x) <= TOL_FIELD, (f, j)


def test_filter_full_size_largest_scales_properties(full, oracle_mesh):
    """The longest solves (l up to 1000 h, ~1e4 iterations): true residual through if_apply, mean conservation,
    energy identity phi^T M x = x^T A_l x >= x^T M x.  The oracle would need minutes per solve here."""
    import torch
    lib, w, h = full
    ells = w.ells[-8:]
    out, st = lib.if_filter(h, w.fields, ells, 1)
    assert st["code"] == 0 and st["iters"].max() > 2000
    area = torch.from_numpy(oracle_mesh.area()).to(out.device)
    fields = torch.from_numpy(w.fields).to(out.device)
    for f, j in ((0, 7), (1, 7), (0, 0)):
        x = out[f, j]
        b = area * fields[f]
        ax = lib.if_apply(h, x[None, :], ells[j:j + 1], 1)[0, 0]
        true_res = float(torch.linalg.norm(b - ax) / torch.linalg.norm(b))
        assert true_res <= 1e-9, (f, j, true_res)                        # recursive 1e-12; true floors near u*kappa
        mean_in, mean_out = float((area * fields[f]).sum()), float((area * x).sum())
        assert abs(mean_out - mean_in) <= 1e-9 * float((area * fields[f].abs()).sum())
        lhs, mid, low = float((b * x).sum()), float((x * ax).sum()), float((area * x * x).sum())
        assert abs(lhs - mid) <= 1e-8 * abs(lhs) and mid >= low * (1 - 1e-12)


def test_multigrid_spectrum_full_size(full, oracle_mesh, jacobi_spectrum):
    """solver = 1 (smoothed-aggregation preconditioner on the scales >= 4 mean edges, Jacobi below) on the bench
    step: the same energies as the Jacobi-preconditioned run, an order of magnitude fewer iterations on the large
    scales, and the true residual of the largest scale through if_apply."""
    import torch
    lib, w, h = full
    sp = lib.if_spectrum(h, w.fields, w.ells, 1, solver=1, mg_min_ell=4.0)
    st, stj = sp["stats"], jacobi_spectrum["stats"]
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["rel_res"] <= 1e-12)
    assert np.all(np.abs(sp["energy"] - jacobi_spectrum["energy"]) <= 1e-9 * jacobi_spectrum["energy"])
    assert np.all(np.diff(sp["energy"], axis=1) < 0.0) and np.all(sp["E"] > 0.0)
    big = w.ells >= 4.0 * h.mean_edge
    assert int(big.sum()) * 2 % 16 == 0                                  # whole batches: no remainder moved
    assert st["iters"][:, big].max() < 100 and stj["iters"][:, big].max() > 5000
    assert np.array_equal(st["iters"][:, ~big] > 0, stj["iters"][:, ~big] > 0)
    assert np.all(np.abs(st["iters"][:, ~big] - stj["iters"][:, ~big]) <= 2)     # small scales: the Jacobi path
    assert st["rhs_iters"] < 0.02 * stj["rhs_iters"]
    for f, j in ((0, 16), (1, 12)):                                      # multigrid-solved, oracle in seconds
        x, info = oracle_mesh.solve(w.fields[f], float(w.ells[j]), 1)
        assert info["status"] == 0 and big[j]
        e = oracle_mesh.energy(x)
        assert abs(sp["energy"][f, j] - e) <= TOL_BIN * e, (f, j)
    out, sf = lib.if_filter(h, w.fields[:1], w.ells[-1:], 1, solver=1)
    assert sf["code"] == 0 and sf["iters"].max() < 100
    area = torch.from_numpy(oracle_mesh.area()).to(out.device)
    b = area * torch.from_numpy(w.fields[0]).to(out.device)
    ax = lib.if_apply(h, out[0, 0][None, :], w.ells[-1:], 1)[0, 0]
    assert float(torch.linalg.norm(b - ax) / torch.linalg.norm(b)) <= 1e-9
    assert abs(float((area * out[0, 0]).sum()) - float(b.sum())) <= 1e-9 * float(b.abs().sum())


# ------------------------------------------------------------------------------------------ the other full-size configs
def test_config2_full_size_sampled(oracle_mod):
    """Config 2 at full size (512 x 512 jittered periodic grid with slivers, 2 fields x 20 scales): all 40 solves
    on the GPU, a sample of them (including the largest scale of each field) against the oracle."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2404_07398_b200 as lib
    w = make_config(2)
    assert w.mesh.n_vert == 262144 and w.n_rhs == 40
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    h = lib.if_prepare(w.mesh.coords, w.mesh.tri, w.mesh.period)
    assert h.unstaged_tiles == 0                      # 2-D Morton order: every tile staged in shared memory
    out, st = lib.if_filter(h, w.fields, w.ells, 1)
    sp = lib.if_spectrum(h, w.fields, w.ells, 1)
    assert st["code"] == 0 and sp["stats"]["code"] == 0
    assert np.all(np.diff(sp["energy"], axis=1) < 0.0)
    for f, j in ((0, 0), (1, 6), (0, 12), (0, 19), (1, 19)):
        x, info = om.solve(w.fields[f], float(w.ells[j]), 1)
        assert info["status"] == 0
        assert rel(out[f, j].cpu().numpy(), x) <= TOL_FIELD, (f, j)
        e = om.energy(x)
        assert abs(sp["energy"][f, j] - e) <= TOL_BIN * e, (f, j)
    h.close()


def n2_true_residual_bound(ell_over_h):
    """Largest TRUE relative residual accepted for an n = 2 solve that converged to a recursive 1e-12: the true residual
    floors near u kappa, kappa ~ 1/2 (l^2 lambda_max)^2 ~ l^4 (the oracle records 1e-10 at 8 h,
    1e-9 to 3e-9 at 16 h, 1.5e-8 to 4.6e-8 at 32 h): 2e-7 (l / 32 h)^4 + 1e-10."""
    return 2e-7 * (ell_over_h / 32.0) ** 4 + 1e-10


def test_config3_full_size_biharmonic_all_scales(oracle_mod):
    """Config 3 at full size (icosphere level 9, n = 2), ALL 20 scales 1 ... 32 h through the multigrid product
    preconditioner (solver = 1): the three smallest scales against the oracle (it needs minutes beyond l ~ 2 h), every
    scale through its true residual (if_apply), mean conservation and the energy identity; the Jacobi path on the
    scales it finishes in seconds gives the same fields."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2404_07398_b200 as lib
    w = make_config(3)
    assert w.mesh.n_vert == 2621442 and w.order_n == 2 and w.n_rhs == 20
    assert abs(w.ells[-1] / w.mesh.h - 32.0) < 1e-9
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, None)
    h = lib.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=lib.IF_FLAG_MULTIGRID)
    out, st = lib.if_filter(h, w.fields, w.ells, 2, solver=1)
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["rel_res"] <= 1e-12)
    assert st["mg_batch_iters"] > 0 and st["iters"].max() < 150          # Jacobi-PCG: 64 000 at 32 h
    sp = lib.if_spectrum(h, w.fields, w.ells, 2, solver=1)
    assert sp["stats"]["code"] == 0 and np.all(np.diff(sp["energy"], axis=1) < 0.0) and np.all(sp["E"] > 0.0)
    for j in (0, 1, 2):
        x, info = om.solve(w.fields[0], float(w.ells[j]), 2)
        assert info["status"] == 0
        assert rel(out[0, j].cpu().numpy(), x) <= TOL_FIELD, j
        e = om.energy(x)
        assert abs(sp["energy"][0, j] - e) <= TOL_BIN * e, j
    area = torch.from_numpy(om.area()).to(out.device)
    phi = torch.from_numpy(w.fields[0]).to(out.device)
    b = area * phi
    for j in range(20):
        x = out[0, j]
        ax = lib.if_apply(h, x[None, :], w.ells[j:j + 1], 2)[0, 0]
        res = float(torch.linalg.norm(b - ax) / torch.linalg.norm(b))
        assert res <= n2_true_residual_bound(w.ells[j] / w.mesh.h), (j, res)
        assert abs(float((area * x).sum()) - float(b.sum())) <= 1e-9 * float(b.abs().sum())
        lhs, mid, low = float((b * x).sum()), float((x * ax).sum()), float((area * x * x).sum())
        assert abs(lhs - mid) <= 1e-6 * abs(lhs) and mid >= low * (1 - 1e-12)
        e_j = 0.5 * low / float(area.sum())
        assert abs(e_j - sp["energy"][0, j]) <= 1e-9 * e_j
    jac, sj = lib.if_filter(h, w.fields, w.ells[:6], 2)                  # Jacobi-PCG, l <= 2.5 h
    assert sj["code"] == 0
    for j in range(6):
        assert float(torch.linalg.norm(jac[0, j] - out[0, j]) / torch.linalg.norm(jac[0, j])) <= 1e-9
    h.close()


# the right-hand sides of config 5 that are checked one by one: field 0 at every 4th scale, every
# other field at the first, the middle and the last scale
CFG5_SUBSET = [(0, j) for j in range(0, 40, 4)] + [(f, j) for f in range(1, 8) for j in (0, 20, 39)]
CFG5_ORACLE = [(0, 0), (0, 4), (3, 0), (7, 0)]            # of those, against the oracle (l <= 1.43 h: seconds to a minute)


def test_config5_full_size_all_320_right_hand_sides(full, oracle_mesh, oracle_mod):
    """Config 5 = config 4's mesh (ONE if_prepare), 8 fields x 40 scales = 320 right-hand sides, n = 2, 16 columns per
    SpMM, l = 1 ... 32 h, in the launch configuration bench.py --config 5 times (if_spectrum, solver = 1).  All 320
    converge; energies monotone per field; the 31 right-hand sides of CFG5_SUBSET are solved again by if_filter and
    checked by their true residual, mean conservation and their energy against the spectrum call; CFG5_ORACLE
    against the oracle element by element."""
    import torch
    lib, w4, h = full
    w = make_config(5)
    assert w.fields.shape == (8, w4.mesh.n_vert) and w.order_n == 2 and np.array_equal(w.mesh.tri, w4.mesh.tri)
    assert w.ells.shape[0] == 40 and abs(w.ells[-1] / w.mesh.h - 32.0) < 1e-9
    sp = lib.if_spectrum(h, w.fields, w.ells, 2, solver=1)
    st = sp["stats"]
    assert st["code"] == 0 and st["iters"].shape == (8, 40) and np.all(st["status"] == 0)
    assert np.all(st["rel_res"] <= 1e-12) and st["iters"].max() < 150 and st["mg_batch_iters"] > 0
    assert np.all(np.diff(sp["energy"], axis=1) < 0.0) and np.all(sp["E"] > 0.0)
    scales = sorted({j for _, j in CFG5_SUBSET})
    out, sf = lib.if_filter(h, w.fields, w.ells[scales], 2, solver=1)
    assert sf["code"] == 0
    area = torch.from_numpy(oracle_mesh.area()).to(out.device)
    tot = float(area.sum())
    for f, j in CFG5_SUBSET:
        x = out[f, scales.index(j)]
        b = area * torch.from_numpy(w.fields[f]).to(out.device)
        ax = lib.if_apply(h, x[None, :], w.ells[j:j + 1], 2)[0, 0]
        res = float(torch.linalg.norm(b - ax) / torch.linalg.norm(b))
        assert res <= n2_true_residual_bound(w.ells[j] / w.mesh.h), (f, j, res)
        assert abs(float((area * x).sum()) - float(b.sum())) <= 1e-9 * float(b.abs().sum())
        e = 0.5 * float((area * x * x).sum()) / tot
        assert abs(e - sp["energy"][f, j]) <= 1e-8 * e, (f, j)
    for f, j in CFG5_ORACLE:
        x, info = oracle_mesh.solve(w.fields[f], float(w.ells[j]), 2)
        assert info["status"] == 0
        assert rel(out[f, scales.index(j)].cpu().numpy(), x) <= TOL_FIELD, (f, j)
        e = oracle_mesh.energy(x)
        assert abs(sp["energy"][f, j] - e) <= TOL_BIN * e, (f, j)


def test_vector_filter_large_band(oracle_mod):
    """The coupled vector filter (IF_FLAG_VECTOR) on a latitude band of the level-9 icosphere (2.5 M
    vertices), 4 (u, v) pairs x 6 scales, n = 1, K = 16 (8 pairs per SpMM): one pair at the two smallest scales against
    the oracle's joint PCG, every solve through its true residual (IF_FLAG_TRUE_RESIDUAL); prints the bandwidth of the
    vector kernel A (6 vectors + 20 B per matrix entry + 16 B per row)."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2404_07398_b200 as lib
    from workloads import icosphere, jitter_sphere, log_spaced, sphere_band, sphere_velocity_field
    mesh = sphere_band(jitter_sphere(icosphere(9), 0.25, np.random.default_rng(41)), 70.0)
    rng = np.random.default_rng(42)
    fields = np.empty((8, mesh.n_vert))
    for p in range(4):
        fields[2 * p], fields[2 * p + 1] = sphere_velocity_field(mesh.coords, 200, 64, rng)
    ells = mesh.h * log_spaced(1.0, 24.0, 6)
    VEC = lib.IF_FLAG_VECTOR
    h = lib.if_prepare(mesh.coords, mesh.tri, None, flags=VEC, radius=1.0)
    assert h.n_vert > 2_400_000
    out, st = lib.if_filter(h, fields, ells, 1, flags=VEC | lib.IF_FLAG_TRUE_RESIDUAL)
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["true_res"] <= 1e-10)
    assert np.array_equal(st["iters"][0::2], st["iters"][1::2])          # a pair shares its iteration count
    om = oracle_mod.OracleMesh(mesh.coords, mesh.tri, None)
    om.build_vector(1.0)
    for j in (0, 1):
        xu, xv, info = om.solve_vector(fields[0], fields[1], float(ells[j]), 1)
        assert info["status"] == 0
        assert rel(out[0, j].cpu().numpy(), xu) <= TOL_FIELD and rel(out[1, j].cpu().numpy(), xv) <= TOL_FIELD, j
    sp = lib.if_spectrum(h, fields, ells, 1, flags=VEC | lib.IF_FLAG_PAIRS)
    assert sp["energy"].shape == (4, 6) and np.all(np.diff(sp["energy"], axis=1) < 0.0) and np.all(sp["E"] > 0.0)
    s = sp["stats"]
    if s["kernel_samples"] > 0:
        nbytes = h.n_vert * 16 * 8 * 6 + (h.nnz - h.n_vert) * 20 + h.n_vert * 16
        print(f"vector kernel A: {1e3 * s['spmm_seconds']:.3f} ms per launch, {nbytes / s['spmm_seconds'] / 1e9:.0f} GB/s "
              f"algorithmic ({s['kernel_samples']} samples, V = {h.n_vert})")
    h.close()


def test_vector_filter_large_band_multigrid():
    """The vector filter through the multigrid path (solver = 1: the scalar hierarchy preconditions the coupled system,
    smoothing on the mesh with the metric terms) on the same band, 8 (u, v) pairs x 12 scales from 1 to 400 edge lengths
    -- scales Jacobi-PCG needs thousands of iterations for: every solve through its true residual
    (IF_FLAG_TRUE_RESIDUAL), the small scales against the Jacobi path, kinetic-energy spectra of both paths."""
    import time
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2404_07398_b200 as lib
    from workloads import icosphere, jitter_sphere, log_spaced, sphere_band, sphere_velocity_field
    mesh = sphere_band(jitter_sphere(icosphere(9), 0.25, np.random.default_rng(41)), 70.0)
    rng = np.random.default_rng(42)
    fields = np.empty((16, mesh.n_vert))
    for p in range(8):
        fields[2 * p], fields[2 * p + 1] = sphere_velocity_field(mesh.coords, 200, 64, rng)
    ells = mesh.h * log_spaced(1.0, 400.0, 12)
    VEC = lib.IF_FLAG_VECTOR
    h = lib.if_prepare(mesh.coords, mesh.tri, None, flags=VEC | lib.IF_FLAG_MULTIGRID, radius=1.0)
    out, st = lib.if_filter(h, fields, ells, 1, flags=VEC | lib.IF_FLAG_TRUE_RESIDUAL, solver=1)
    assert st["code"] == 0 and np.all(st["status"] == 0) and np.all(st["true_res"] <= 1e-10), st["true_res"].max()
    assert st["mg_batch_iters"] == st["batch_iters"] > 0
    assert np.array_equal(st["iters"][0::2], st["iters"][1::2])
    jac, sj = lib.if_filter(h, fields[:4], ells[:5], 1, flags=VEC)                      # up to 9 edge lengths
    assert sj["code"] == 0
    assert float((out[:4, :5] - jac).abs().max()) <= 1e-8 * float(jac.abs().max())
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    sp = lib.if_spectrum(h, fields, ells, 1, flags=VEC | lib.IF_FLAG_PAIRS, solver=1)
    t_mg = time.perf_counter() - t0
    assert sp["energy"].shape == (8, 12) and np.all(np.diff(sp["energy"], axis=1) < 0.0) and np.all(sp["E"] > 0.0)
    o = out.cpu().numpy()
    area = lib.if_mesh_export_csr(lib.if_prepare(mesh.coords, mesh.tri, None, flags=lib.IF_FLAG_KEEP_CSR))[3]
    ke = 0.5 * ((area * o[0::2] ** 2).sum(-1) + (area * o[1::2] ** 2).sum(-1)) / area.sum()
    assert np.all(np.abs(sp["energy"] - ke) <= 1e-9 * ke)
    s = sp["stats"]
    print(f"vector filter, multigrid path: V = {h.n_vert}, 8 pairs x 12 scales (1 ... 400 h) in {t_mg:.3f} s, "
          f"{int(s['iters'][0::2].sum())} pair-iterations ({int(s['iters'].min())}-{int(s['iters'].max())} per solve), "
          f"{s['mg_batch_iters']} fused iterations; Jacobi-PCG at 9 h: {int(sj['iters'][:, -1].max())} iterations")
    h.close()
