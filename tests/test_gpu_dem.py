"""GPU parity: CUDA DEM pipeline (through the C ABI) vs the CPU oracle.
north_star: cell ordering and contact pair list bit-exact; per-particle forces after one step
within 1e-12 relative; trajectories over 10 steps within 1e-9."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


PATHS = {"one_launch": {}, "chain_radix": {"no_single_block": 1, "cell_order": 1},
         "chain_counting": {"no_single_block": 1, "cell_order": 2}}


@pytest.fixture(autouse=True, params=list(PATHS))
def dem_path(request):
    """Every test of this file runs on every path of the step: small systems (n <= 4 096) by the single-launch cluster
    kernel, and the chain of kernels that larger systems take with the order by cell from the radix passes and from
    the counting sort (ledds_dem_params.no_single_block, cell_order)."""
    from paper_2512_04997_b200 import Dem
    old = Dem.DEFAULTS
    Dem.DEFAULTS = PATHS[request.param]
    yield request.param
    Dem.DEFAULTS = old


def both(pd, x, v, w, R):
    import oracle
    from paper_2512_04997_b200 import Dem
    return oracle.Dem(pd, x, v, w, R), Dem(pd, x, v, w, R)


def check_state(o, g, steps_done, box):
    q = g.query()
    assert q["status"] == 0
    assert np.array_equal(q["key"], o.key[o.idx]) and np.array_equal(q["idx"], o.idx)
    assert np.array_equal(q["pairs"], o.pairs), (len(q["pairs"]), len(o.pairs))
    fs = max(np.abs(o.F).max(), 1e-300)
    assert np.abs(q["F"] - o.F).max() <= 1e-12 * fs
    assert np.abs(q["M"] - o.M).max() <= 1e-12 * max(np.abs(o.M).max(), 1e-300)
    if len(o.pairs):
        assert np.abs(q["pair_dt"] - o.dt_hist).max() <= 1e-12 * max(np.abs(o.dt_hist).max(), 1e-300)
    s = g.state()
    assert np.abs(s["x"] - o.x).max() <= 1e-9 * box
    assert np.abs(s["v"] - o.v).max() <= 1e-9 * max(np.abs(o.v).max(), 1e-300)
    assert np.abs(s["w"] - o.w).max() <= 1e-9 * max(np.abs(o.w).max(), 1e-300)


@pytest.mark.parametrize("seed,bc,n", [(1, (1, 1, 1), 3000), (2, (0, 0, 0), 4000), (3, (0, 1, 0), 1777), (4, (1, 0, 1), 33)])
def test_random_overlapping_cloud(seed, bc, n):
    # dense random polydisperse cloud: many contacts, friction, rotation, periodic wrap, walls
    pd, x, v, w, R = W.dem_random(seed, n, box=(14.0, 11.0, 9.0), bc=bc)
    pd["max_contacts"] = 32
    o, g = both(pd, x, v, w, R)
    check_state(o, g, 0, 14.0)                                 # forces of the initial state, a(0)
    assert np.abs(g.state()["a"] - o.a).max() <= 1e-12 * np.abs(o.a).max()
    o.step(); g.step()
    check_state(o, g, 1, 14.0)                                 # forces after one step: 1e-12
    for _ in range(9):
        o.step(); g.step()
    check_state(o, g, 10, 14.0)                                # trajectories over 10 steps: 1e-9


def test_config1_gas_full():
    # BASELINE configs[0] at full size: 2048 spheres, 10 steps, then 200 more with ordering still exact
    pd, x, v, w, R = W.cfg1_gas()
    o, g = both(pd, x, v, w, R)
    o.step(10); g.step(10)
    check_state(o, g, 10, pd["hi"][0])


def test_multi_tile_sort_and_ragged_tail():
    # 70 001 particles: 18 sort tiles with a ragged last tile, 3 radix passes (grid has > 65536 cells)
    n_side = 42
    pd, x, v, w, R = W.cfg5_pour(seed=9, n_side=n_side, n_part=70001, dense=True)
    o, g = both(pd, x, v, w, R)
    check_state(o, g, 0, pd["hi"][2])
    assert len(o.pairs) > 50000
    o.step(2); g.step(2)
    check_state(o, g, 2, pd["hi"][2])


def test_edge_cases_single_particle_and_no_contacts():
    pd = W.dem_defaults(1, (0, 0, 0), (4, 4, 4), (1, 1, 1), cell=1.0, dt=1e-3, g=(0, 0, -9.81), density=1000.0, kn=1e5,
                        restitution=0.5, mu=0.3)
    o, g = both(pd, [[2, 2, 0.45]], [[0.1, 0, 0]], [[0, 0, 0]], [0.5])
    o.step(20); g.step(20)
    check_state(o, g, 20, 4.0)
    assert o.pairs.tolist() == [[0, 5]]
    # no contact at all
    pd, x, v, w, R = W.cfg5_pour(seed=3, n_side=10, n_part=1000, dense=False)
    o, g = both(pd, x, v, w, R)
    o.step(3); g.step(3)
    check_state(o, g, 3, pd["hi"][2])
    assert len(o.pairs) == 0


def test_contact_slot_overflow_is_flagged():
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Dem
    pd, x, v, w, R = W.dem_random(5, 400, box=(3.0, 3.0, 3.0))
    pd["max_contacts"] = 2
    g = Dem(pd, x, v, w, R)
    assert int(g.status[0].item()) & L.ST_CONTACT_OVERFLOW


def test_history_persists_and_is_dropped():
    # oblique wall impact: tangential history accumulates during the contact, gone afterwards
    pd = W.dem_defaults(1, (0, 0, 0), (10, 1, 1), (1, 1, 1), cell=0.2, dt=2e-5, g=(0, 0, 0), density=2000.0, kn=1e6,
                        restitution=1.0, mu=0.3)
    o, g = both(pd, [[1.0, 0.5, 0.05 + 1e-6]], [[2.0, 0, -1.0]], [[0, 0, 0]], [0.05])
    seen = 0
    for _ in range(200):
        o.step(); g.step()
        q = g.query()
        assert np.array_equal(q["pairs"], o.pairs)
        if len(o.pairs):
            seen += 1
            assert np.abs(q["pair_dt"] - o.dt_hist).max() <= 1e-12 * np.abs(o.dt_hist).max()
    assert seen > 10 and len(o.pairs) == 0
    s = g.state()
    assert np.abs(s["w"] - o.w).max() <= 1e-9 * np.abs(o.w).max() and abs(o.w[0, 1]) > 1.0


def test_full_size_config5_dense_state():
    # BASELINE configs[4] size (4 000 000 polydisperse spheres) in the supplementary dense state, launch
    # configuration of bench.py: ordering, pair list and contact forces of the initial state against the oracle
    pd, x, v, w, R = W.cfg5_pour(dense=True)
    o, g = both(pd, x, v, w, R)
    check_state(o, g, 0, pd["hi"][2])
    assert len(o.pairs) > 5_000_000


def test_full_size_config5_pour_ordering_after_steps():
    # the dilute pour state at full size: 3 steps on the GPU, then the ordering must be the stable argsort of the
    # keys of the GPU's own positions (host-side check of a5-a7 at a size the oracle does not step quickly)
    import oracle
    pd, x, v, w, R = W.cfg5_pour()
    from paper_2512_04997_b200 import Dem
    g = Dem(pd, x, v, w, R)
    g.step(3)
    q = g.query()
    nc, inv_h = oracle.dem_grid(pd)
    xs = g.state()["x"]
    c = np.clip(np.floor((xs - np.asarray(pd["lo"])) * inv_h).astype(np.int64), 0, np.asarray(nc) - 1)
    key = (c[:, 0] + nc[0] * (c[:, 1] + nc[1] * c[:, 2])).astype(np.uint32)
    idx = np.argsort(key, kind="stable").astype(np.uint32)
    assert np.array_equal(q["idx"], idx) and np.array_equal(q["key"], key[idx])
    assert q["status"] == 0 and len(q["pairs"]) == 0
    # free fall so far: every sphere has v_z = -g t exactly as integrated (Eq. 18), no contact yet
    assert np.allclose(g.state()["v"][:, 2], -9.81 * 3 * pd["dt"], rtol=1e-12)


@pytest.mark.parametrize("seed,bc,n", [(11, (1, 1, 1), 2500), (12, (0, 1, 0), 1500)])
def test_hertz_mindlin_cloud(seed, bc, n):
    # PAPER.md:968-1001 (A.1)-(A.8): stiffness and damping per contact from Young's modulus, Poisson ratio and the
    # overlap; walls of another material; polydisperse radii, friction, rotation, periodic wrap
    pd, x, v, w, R = W.dem_random(seed, n, box=(14.0, 11.0, 9.0), bc=bc)
    pd.update(max_contacts=32, model=1, young=2.0e6, poisson=0.3, young_w=7.0e6, poisson_w=0.22, dt=2e-5)
    o, g = both(pd, x, v, w, R)
    check_state(o, g, 0, 14.0)
    o.step(); g.step()
    check_state(o, g, 1, 14.0)
    for _ in range(9):
        o.step(); g.step()
    check_state(o, g, 10, 14.0)


@pytest.mark.parametrize("bc", [(1, 1, 1), (0, 0, 0)])
def test_first_look_in_single_precision_never_hides_a_contact(bc):
    # The detect kernel looks at a candidate first on single-precision records (dem_near) and only then decides
    # Eq. (2) in double.  Here single precision cannot tell the pairs apart: a 300^3 box of unit cells with
    # spheres of radius ~1e-3 (coordinate rounding 300 * 2^-24 = 1.8 % of a radius) whose partner sits at
    # (R_i + R_j)(1 +- 1e-12 ... 1e-4), some of them across a periodic face; one particle far outside the box
    # (NaN record).  The pair list must still equal the oracle's (which is pinned to the O(N^2) list).
    g = np.random.Generator(np.random.PCG64(77))
    npair = 1500
    L = 300.0
    R = g.uniform(0.8e-3, 1.2e-3, 2 * npair + 1)
    a = g.uniform(1.0, L - 1.0, (npair, 3))
    a[:200, 0] = g.uniform(0.0, 2.0e-4, 200)                   # next to the x = 0 face: the partner wraps or meets the wall
    e = g.normal(size=(npair, 3)); e /= np.linalg.norm(e, axis=1)[:, None]
    e[:200, 0] = -np.abs(e[:200, 0])
    gap = np.where(g.random(npair) < 0.5, -1.0, 1.0) * 10.0 ** g.uniform(-12, -4, npair)
    b = a + e * ((R[:npair] + R[npair:2 * npair]) * (1.0 + gap))[:, None]
    x = np.concatenate([a, b, [[L + 450.0, 10.0, 10.0]]])      # the last one has left the box
    if bc == (0, 0, 0):
        x[:-1] = np.mod(x[:-1], L)
    else:
        x[:-1] = np.clip(x[:-1], 0.0, L)
    pd = W.dem_defaults(len(R), (0, 0, 0), (L, L, L), bc, cell=1.0, dt=1e-7, g=(0, 0, 0), density=1000.0, kn=1e2,
                        restitution=0.8, mu=0.4)
    v = np.zeros_like(x); w = np.zeros_like(x)
    o, gp = both(pd, x, v, w, R)
    q = gp.query()
    assert np.array_equal(q["idx"], o.idx)
    assert np.array_equal(q["pairs"], o.pairs), (len(q["pairs"]), len(o.pairs))
    touching = int((o.pairs[:, 1] < len(R)).sum())
    assert 400 < touching < npair - 400                        # both outcomes are well represented


@pytest.mark.parametrize("model,eps_w", [(0, 0.5), (0, 0.8), (1, 0.5)])
def test_wall_bounce_with_damping(model, eps_w):
    # reading G13: wall contact with its own stiffness, restitution and material, m* = m_i, R* = R_i
    # (pinned for the oracle by restitution = eps_w and the Hertz impact depth, tests/test_oracle_dem.py): a sphere
    # thrown obliquely at the floor with spin, followed through the whole contact
    R, rho = 0.5e-3, 2500.0
    m = rho * 4.0 / 3.0 * np.pi * R ** 3
    kn_w = 2.0e4
    tc = np.pi / np.sqrt(kn_w / m)
    pd = W.dem_defaults(1, (0, 0, 0), (1, 1, 1), (1, 1, 1), cell=0.5, dt=tc / 60.0, g=(0, 0, -9.81), density=rho, kn=1.0e4,
                        restitution=1.0, mu=0.0, kn_w=kn_w, kt_w=kn_w * 2 / 7, restitution_w=eps_w, mu_w=0.4, model=model,
                        young=1.0e7, poisson=0.3, young_w=4.0e7, poisson_w=0.2)
    o, g = both(pd, [[0.5, 0.5, R * (1 + 1e-3)]], [[0.03, -0.01, -0.1]], [[5.0, -3.0, 2.0]], [R])
    seen = 0
    for _ in range(60):
        o.step(10); g.step(10)
        check_state(o, g, 0, 1.0)
        seen += len(o.pairs)
        if seen and not len(o.pairs):
            break
    assert seen >= 3 and len(o.pairs) == 0 and o.v[0, 2] > 0.3 * eps_w * 0.1


def test_input_contract_violations_are_flagged():
    # a sphere wider than a grid cell (contacts beyond the 27-cell walk would be missed) and a centre outside
    # a walled box (cell index clamped) raise status bits instead of passing silently
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Dem
    pd = W.dem_defaults(3, (0, 0, 0), (4, 4, 4), (1, 1, 0), cell=1.0, dt=1e-4, g=(0, 0, 0), density=1000.0, kn=1e5,
                        restitution=0.5, mu=0.3)
    x = np.array([[1.0, 1.0, 1.0], [3.0, 3.0, 3.0], [2.0, 2.0, 2.0]])
    z = np.zeros((3, 3))
    g = Dem(pd, x, z, z, np.array([0.3, 0.5, 0.4]))
    assert int(g.status[0].item()) == 0                        # 2 R = cell is allowed
    g = Dem(pd, x, z, z, np.array([0.3, 0.51, 0.4]))
    assert int(g.status[0].item()) == L.ST_RADIUS_RANGE
    x[0, 1] = 4.2                                              # outside the walled y range
    g = Dem(pd, x, z, z, np.array([0.3, 0.5, 0.4]))
    assert int(g.status[0].item()) & L.ST_OUT_OF_BOX
    x[0, 1] = 1.0; x[0, 2] = 4.2                               # z is periodic: wrapped by the drift, never out of the box
    g = Dem(pd, x, z, z, np.array([0.3, 0.5, 0.4]))
    g.step(1)
    assert int(g.status[0].item()) == 0


def test_sort_is_skipped_only_when_it_is_the_identity():
    # the radix passes of a step return at once when the keys are still in order (ledds.h: sort_every_step).  Fast
    # particles (a few change their cell every step) and a frozen state, each with the skip and with the passes forced:
    # ordering, pair list and state must be the oracle's / bit-identical between the two settings
    from paper_2512_04997_b200 import Dem
    import oracle
    pd, x, v, w, R = W.dem_random(21, 2000, box=(14.0, 11.0, 9.0), bc=(0, 1, 0))
    pd["max_contacts"] = 32
    for scale in (40.0, 0.0):
        vv = v * scale
        o = oracle.Dem(pd, x, vv, w, R)
        g0, g1 = Dem(pd, x, vv, w, R), Dem(dict(pd, sort_every_step=1), x, vv, w, R)
        crossed = 0
        for _ in range(8):
            key_before = o.key.copy()
            o.step(); g0.step(); g1.step()
            crossed += int((o.key != key_before).sum())
            q0, q1 = g0.query(), g1.query()
            assert np.array_equal(q0["idx"], o.idx) and np.array_equal(q0["key"], o.key[o.idx])
            assert np.array_equal(q0["pairs"], o.pairs)
            for k in ("idx", "key", "pairs", "pair_dt", "F", "M"):
                assert np.array_equal(q0[k], q1[k]), k
            s0, s1 = g0.state(), g1.state()
            assert all(np.array_equal(s0[k], s1[k]) for k in s0)
        assert (crossed > 20) if scale else (crossed < 20)
