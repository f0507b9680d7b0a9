"""CPU checks of bench.py's byte models (pure functions): the Jacobi iteration's 78.5 B per row and right-hand side and
the multigrid iteration's groups for a hierarchy shaped like config 4's (DESIGN.md sections 5 and 9g)."""
import bench


def test_jacobi_iteration_bytes():
    V, nnz, K = 7340033, 51300000, 16
    ab = bench.algorithmic_bytes(V, nnz, K, 1)
    per = ab["iteration"] / (V * K)
    assert 78.0 < per < 79.0                       # 72 B of vectors + 6.5 B of matrix per row and right-hand side
    assert ab["spmm"] == V * K * 48 + (nnz - V) * 12 + V * 16 and ab["update"] == V * K * 24 + V * 16
    ab2 = bench.algorithmic_bytes(V, nnz, K, 2)
    assert ab2["spmm"] - ab["spmm"] == V * K * 24 + (nnz - V) * 12 + V * 16     # second pass: t, p' in, q out + matrix


def test_multigrid_iteration_bytes():
    V, nnz = 7340033, 51300000
    info = {"levels": 6, "rows": [V, 814852, 80749, 7379, 668, 64], "nnz": [nnz, 10185650, 1695729, 212515, 22311, 1837],
            "p_nnz": [19084086, 2933467, 379520, 42060, 4075, 0], "sweeps": {1: [1, 1, 2], 2: [4, 2, 2]}}
    vec = V * 128
    matrix = (nnz - V) * 12 + V * 16
    g1 = bench.mg_algorithmic_bytes(V, nnz, info, 1)
    assert g1["A"] == 6 * vec + matrix and g1["MGR"] == 4 * vec + matrix and g1["last"] == 3 * vec + matrix
    assert g1["iteration"] == sum(v for k, v in g1.items() if k != "iteration")
    assert 19.0e9 < g1["iteration"] < 20.5e9                       # 19.8 GB on config 4
    assert g1["level1"] > 10 * g1["coarse"] / 3                    # level 1 dominates the coarse part
    g2 = bench.mg_algorithmic_bytes(V, nnz, info, 2)
    assert g2["A"] == 9 * vec + 2 * matrix and g2["MGR"] == 6 * vec + 2 * matrix
    assert g2["last"] == 2 * 7 * (3 * vec + matrix)                # two cycles x (2 sweeps + residual + 4 sweeps)
    assert g2["iteration"] > 3.5 * g1["iteration"]
