"""The entry point that allocates nothing (if_energy_noalloc: scratch in a static device array, paper_2404_07398_b200/csrc/
noalloc.cu) against the existing path: the energies if_spectrum reports for the same filtered fields, and the plain
definition evaluated with torch on the device.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu

TOL_BIN = 1e-6      # the tolerance the other tests put on energies / spectrum bins (BASELINE.json north_star)


def test_energy_noalloc_matches_the_existing_path_twice_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2404_07398_b200 as ifl
    ifl.load_library()
    w = make_config(4, level=6, n_ells=8)                      # 28 673 vertices: 113 blocks of the reduction grid
    h = ifl.if_prepare(w.mesh.coords, w.mesh.tri, None, flags=ifl.IF_FLAG_KEEP_CSR)
    sp = ifl.if_spectrum(h, w.fields, w.ells, 1)                 # existing path: energies inside the solve call
    out, st = ifl.if_filter(h, w.fields, w.ells, 1)              # the same filtered fields, [2][8][V] on the device
    assert sp["stats"]["code"] == 0 and st["code"] == 0
    flat = out.reshape(-1, h.n_vert)                             # 16 fields
    area = torch.from_numpy(ifl.if_mesh_export_csr(h)[3]).to(flat.device)
    plain = (0.5 * (area * flat * flat).sum(dim=1) / area.sum()).cpu().numpy()
    e1, e2, e3 = (torch.full((flat.shape[0],), -1.0, dtype=torch.float64, device=flat.device) for _ in range(3))
    part = flat[:5]
    torch.cuda.synchronize()
    allocs = lambda: torch.cuda.memory_stats()["allocation.all.allocated"]      # allocations so far (monotonic)
    before = allocs()
    ifl.if_energy_noalloc(h, flat, out=e1)
    # second call in a row: the shared scratch array holds the first call's partial sums and ticket
    ifl.if_energy_noalloc(h, part, out=e2[:5])
    ifl.if_energy_noalloc(h, flat, out=e3)
    assert allocs() == before                                    # nothing was allocated through torch either
    first, half, second = e1.cpu().numpy(), e2[:5].cpu().numpy(), e3.cpu().numpy()
    want = sp["energy"].reshape(-1)
    for got in (first, second):
        assert np.all(np.abs(got - want) <= TOL_BIN * want), np.abs(got / want - 1).max()
        assert np.all(np.abs(got - plain) <= 1e-12 * plain)
    assert np.array_equal(first, second) and np.array_equal(half, first[:5])      # deterministic, no stale state
    # the fixed maximum: 32 fields per call
    many = flat[:1].expand(33, -1).contiguous()
    with pytest.raises(ifl.ImplicitFilterError) as err:
        ifl.if_energy_noalloc(h, many)
    assert err.value.code == ifl.binding.IF_ELIMIT
    full = ifl.if_energy_noalloc(h, many[:32]).cpu().numpy()
    assert np.all(np.abs(full - want[0]) <= TOL_BIN * want[0])
    # on another stream
    s2 = torch.cuda.Stream()
    s2.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s2):
        third = ifl.if_energy_noalloc(h, flat, out=e1, stream=s2)
    s2.synchronize()
    assert np.array_equal(third.cpu().numpy(), first)
    h.close()
