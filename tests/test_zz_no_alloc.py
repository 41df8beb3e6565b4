"""GPU: ledds_dem_cell_order_static -- the entry point that allocates nothing (its sort scratch is a static device
array inside the library, include/ledds.h) -- against the existing path (ledds_dem_init + ledds_dem_query), bit for
bit (integer work), on calls in a row that share the static array.

Collected last on purpose (pytest orders files by name): the suite runs with pytest -x."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


def existing_path(pd, x, v, w, R):
    from paper_2512_04997_b200 import Dem
    q = Dem(pd, x, v, w, R).query()
    assert q["status"] == 0
    return q["idx"], q["key"]


def static_path(pd, x, out=None):
    import torch
    import paper_2512_04997_b200 as L
    n = int(pd["n"])
    xd = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device="cuda").reshape(n, 3)
    idx, key = out if out is not None else (torch.empty(max(n, 4), dtype=torch.int32, device="cuda"),
                                            torch.empty(max(n, 4), dtype=torch.int32, device="cuda"))
    idx.fill_(-1); key.fill_(-1)
    L.ledds_dem_cell_order_static(L.dem_params(pd), xd, idx, key)
    torch.cuda.synchronize()
    u32 = lambda t: t[:n].cpu().numpy().view(np.uint32)
    return u32(idx), u32(key)


def test_static_scratch_cell_order_equals_the_existing_path_on_calls_in_a_row():
    # 70 001 spheres: 23 sort tiles with a ragged last one, 3 radix passes (more than 65 536 cells);
    # then a smaller, periodic cloud with other keys (2 passes): what the first call left in the array must not matter;
    # then the first again
    a = W.cfg5_pour(seed=9, n_side=42, n_part=70001, dense=True)
    b = W.dem_random(7, 33333, box=(40.0, 33.0, 27.0), bc=(0, 1, 0))
    b[0]["max_contacts"] = 32
    want_a = existing_path(*a)
    want_b = existing_path(*b)
    for pd, x, want in ((a[0], a[1], want_a), (b[0], b[1], want_b), (a[0], a[1], want_a), (a[0], a[1], want_a)):
        idx, key = static_path(pd, x)
        assert np.array_equal(key, want[1])
        assert np.array_equal(idx, want[0])
        # and against the definition: ids ordered by (cell key, id)
        assert np.array_equal(np.sort(idx), np.arange(pd["n"], dtype=np.uint32))
        assert np.all((key[1:] > key[:-1]) | ((key[1:] == key[:-1]) & (idx[1:] > idx[:-1])))


def test_static_scratch_capacity_and_edges():
    import torch
    import paper_2512_04997_b200 as L
    cap = L.ledds_dem_cell_order_static_max_n()
    assert cap == 262144
    # one particle more than the static array holds: refused with a clear message, nothing written
    pd = W.dem_defaults(cap + 1, (0, 0, 0), (64, 64, 64), (1, 1, 1), cell=1.0, dt=1e-3, g=(0, 0, 0), density=1.0, kn=1.0,
                        restitution=0.9, mu=0.0)
    x = torch.zeros(cap + 1, 3, dtype=torch.float64, device="cuda")
    idx = torch.full((cap + 1,), -1, dtype=torch.int32, device="cuda")
    key = torch.full((cap + 1,), -1, dtype=torch.int32, device="cuda")
    with pytest.raises(L.LeddsError, match="exceed the static scratch"):
        L.ledds_dem_cell_order_static(L.dem_params(pd), x, idx, key)
    torch.cuda.synchronize()
    assert int(idx.max()) == -1 and int(key.max()) == -1
    # exactly the maximum, all particles in one cell but the last: ids come back in order
    pd["n"] = cap
    xh = np.full((cap, 3), 0.5)
    xh[-1] = (63.5, 63.5, 63.5)
    i2, k2 = static_path(pd, xh)
    assert np.array_equal(i2, np.arange(cap, dtype=np.uint32))
    assert np.all(k2[:-1] == 0) and k2[-1] == 64 ** 3 - 1
    # empty system: nothing to do, no error
    pd["n"] = 0
    L.ledds_dem_cell_order_static(L.dem_params(pd), None, None, None)
