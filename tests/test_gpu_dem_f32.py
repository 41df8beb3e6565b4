"""GPU parity of the single-precision DEM calls (ledds_dem_*_f32).

The oracle stays fp64.  Discrete results (cell ordering, contact pair list) are decisions of fp32 arithmetic here
(include/ledds.h states the rule); they are checked bit for bit against the same decisions taken in numpy float32 on
the GPU's own positions (numpy's float32 +, -, *, sqrt are the IEEE operations the kernels use: dem.cu is compiled
without FMA contraction).  Continuous results are compared with the fp64 oracle started from the same fp32-rounded
inputs, within bounds derived from the rounding of the arithmetic:
  * overlap delta_n = (R_i + R_j) - |r_i - r_j|: four roundings of quantities of size <= 2 R_max + the rounding of the
    coordinates' difference, so |d delta| <= 8 * 2^-24 * L (L = box size bounds every coordinate); a contact force
    differs by at most k_n * that + 2e-5 |F| (the products with velocities and unit vectors: ~20 roundings);
  * a position gains <= 2 roundings of size 2^-24 L per step; velocities follow from the forces."""
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
EPS32 = 2.0 ** -24
f32 = np.float32


def both32(pd, x, v, w, R):
    import oracle
    from paper_2512_04997_b200 import Dem
    x, v, w, R = (np.asarray(a, f32) for a in (x, v, w, R))
    o = oracle.Dem(pd, x.astype(np.float64), v.astype(np.float64), w.astype(np.float64), R.astype(np.float64))
    return o, Dem(pd, x, v, w, R, precision="f32")


def grid32(pd):
    """the grid of ledds_dem_params in the kernel's fp32 form"""
    lo, hi = np.asarray(pd["lo"], np.float64), np.asarray(pd["hi"], np.float64)
    nc = np.maximum(1, np.floor((hi - lo) / pd["cell"]).astype(np.int64))
    return lo.astype(f32), hi.astype(f32), (hi - lo).astype(f32), nc, (nc / (hi - lo)).astype(f32)


def keys32(pd, x):
    lo, hi, L, nc, inv_h = grid32(pd)
    c = np.floor((x - lo[None, :]) * inv_h[None, :]).astype(np.int64)       # float32 arithmetic
    c = np.clip(c, 0, nc[None, :] - 1)
    return (c[:, 0] + nc[0] * (c[:, 1] + nc[1] * c[:, 2])).astype(np.uint32)


def pairs32(pd, x, R):
    """O(N^2) pair list with every decision taken in float32, in the kernel's operation order"""
    lo, hi, L, nc, inv_h = grid32(pd)
    n = len(R)
    out = []
    for i in range(n):
        d = x[i][None, :] - x[i + 1:]                                       # float32
        for a in range(3):
            if not pd["bc"][a]:
                da = d[:, a]
                da = np.where(da > f32(0.5) * L[a], da - L[a], np.where(da < f32(-0.5) * L[a], da + L[a], da))
                d[:, a] = da
        d2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
        hit = ((R[i] + R[i + 1:]) - np.sqrt(d2)) > 0
        out += [(i, i + 1 + j) for j in np.nonzero(hit)[0]]
        for wl in range(6):
            ax, side = wl >> 1, wl & 1
            if pd["bc"][ax]:
                dist = hi[ax] - x[i, ax] if side else x[i, ax] - lo[ax]
                if R[i] - dist > 0:
                    out.append((i, n + wl))
    return np.asarray(out, np.uint32).reshape(-1, 2)


def check_decisions(pd, g):
    """ordering and pair list of the GPU's current state == the fp32 decisions on its own positions"""
    q = g.query()
    x = g.state()["x"]
    R = g.radius.cpu().numpy()
    assert x.dtype == np.float32 and q["status"] == 0
    key = keys32(pd, x)
    idx = np.argsort(key, kind="stable").astype(np.uint32)
    assert np.array_equal(q["idx"], idx) and np.array_equal(q["key"], key[idx])
    exp = pairs32(pd, x, R)
    assert np.array_equal(q["pairs"], exp), (len(q["pairs"]), len(exp))
    return q


@pytest.mark.parametrize("seed,bc,n", [(1, (1, 1, 1), 2000), (2, (0, 0, 0), 2500), (3, (0, 1, 0), 1333)])
def test_f32_random_cloud_decisions_and_forces(seed, bc, n):
    pd, x, v, w, R = W.dem_random(seed, n, box=(14.0, 11.0, 9.0), bc=bc)
    pd["max_contacts"] = 32
    o, g = both32(pd, x, v, w, R)
    Lbox = 14.0
    q = check_decisions(pd, g)
    # forces of the initial state: the same positions on both sides
    common = len(set(map(tuple, q["pairs"].tolist())) & set(map(tuple, o.pairs.tolist())))
    assert common >= 0.999 * len(o.pairs)                                   # only contacts within rounding of delta_n = 0 differ
    tolF = pd["kn"] * 8 * EPS32 * Lbox + 2e-5 * np.abs(o.F).max()
    assert np.abs(q["F"] - o.F).max() <= tolF
    assert np.abs(q["M"] - o.M).max() <= tolF * float(R.max())
    for _ in range(10):
        o.step(); g.step()
    check_decisions(pd, g)
    s = g.state()
    assert np.abs(s["x"] - o.x).max() <= 4 * 10 * EPS32 * Lbox
    assert np.abs(s["v"] - o.v).max() <= 2e-4 * np.abs(o.v).max()
    assert np.abs(s["w"] - o.w).max() <= 2e-4 * np.abs(o.w).max()


def test_f32_config1_gas_and_multistep_call():
    # BASELINE configs[0] in single precision: 2048 spheres, 50 steps in one call
    pd, x, v, w, R = W.cfg1_gas()
    o, g = both32(pd, x, v, w, R)
    o.step(50); g.step(50)
    check_decisions(pd, g)
    s = g.state()
    Lbox = pd["hi"][0]
    # This gas is stiff (contact time 25 steps) and its dashpot force starts with a jump gamma_n v_n at first touch: a
    # contact that fp32 sees one step before or after fp64 shifts a velocity by gamma_n v_n dt / m ~ 1e-3 m/s and the
    # position by that times the rest of the run; so the bound here is that of a few such events, not of rounding alone
    assert np.abs(s["x"] - o.x).max() <= 1e-4 * Lbox
    assert np.abs(s["v"] - o.v).max() <= 2e-2 * np.abs(o.v).max()
    assert np.sqrt(np.mean((s["x"] - o.x) ** 2)) <= 1e-5 * Lbox


def test_f32_hertz_wall_bounce_and_history():
    # Hertz-Mindlin coefficients, wall contact with friction: the tangential history in fp32
    R, rho = 0.5e-3, 2500.0
    pd = W.dem_defaults(1, (0, 0, 0), (1e-2, 1e-2, 1e-2), (1, 1, 1), cell=2e-3, dt=2e-7, g=(0, 0, -9.81), density=rho, kn=1.0e4,
                        restitution=0.8, mu=0.4, model=1, young=1.0e7, poisson=0.3, young_w=4.0e7, poisson_w=0.2)
    o, g = both32(pd, [[5e-3, 5e-3, R * (1 + 1e-3)]], [[0.03, -0.01, -0.1]], [[5.0, -3.0, 2.0]], [R])
    seen = 0
    for _ in range(60):
        o.step(20); g.step(20)
        q = g.query()
        seen += len(q["pairs"])
        if seen and not len(o.pairs) and not len(q["pairs"]):
            break
    assert seen >= 3
    s = g.state()
    assert np.abs(s["v"] - o.v).max() <= 2e-3 * np.abs(o.v).max()
    assert np.abs(s["w"] - o.w).max() <= 2e-3 * np.abs(o.w).max()


def test_f32_head_on_collision_energy_as_in_the_papers_appendix_b():
    # PAPER.md:559-592 (E1) with its printed parameters, PAPER.md:1003-1023 (Appendix B): elastic head-on collision of two
    # spheres, Hertz contact, R = 150 mm, m = 15.5509 kg, nu = 0.4999, E = 10 MPa, gap 10 um, v = +-0.1 m/s, dt = 1e-4 s,
    # 300 iterations; momentum stays zero and E_k + E_el (Eq. 43-46) is conserved, in fp32 as in fp64 (Fig. B.31 shows the
    # two sets of curves on top of each other)
    from paper_2512_04997_b200 import Dem
    Rs, m, nu, E, gap, v0 = 0.150, 15.5509, 0.4999, 10.0e6, 10.0e-6, 0.1
    rho = m / (4.0 / 3.0 * np.pi * Rs ** 3)
    pd = W.dem_defaults(2, (-1, -1, -1), (1, 1, 1), (1, 1, 1), cell=0.4, dt=1e-4, g=(0, 0, 0), density=rho, kn=1.0, restitution=1.0,
                        mu=0.0, model=1, young=E, poisson=nu)
    x = np.array([[-Rs - gap / 2, 0, 0], [Rs + gap / 2, 0, 0]])
    v = np.array([[v0, 0, 0], [-v0, 0, 0]])
    z = np.zeros((2, 3))
    Ystar, Rstar = E / (2 * (1 - nu * nu)), Rs / 2
    runs = {}
    for prec in ("f64", "f32"):
        g = Dem(pd, x, v, z, np.full(2, Rs), precision=prec)
        en, mom, deepest = [], [], 0.0
        for _ in range(300):
            g.step()
            s = g.state()
            xs, vs = s["x"].astype(np.float64), s["v"].astype(np.float64)
            delta = max(0.0, 2 * Rs - (xs[1, 0] - xs[0, 0]))
            deepest = max(deepest, delta)
            en.append(0.5 * m * (vs ** 2).sum() + 8.0 / 15.0 * Ystar * np.sqrt(Rstar) * delta ** 2.5)
            mom.append(m * vs[:, 0].sum())
        runs[prec] = (np.asarray(en), np.asarray(mom), deepest, vs.copy())
    e0 = m * v0 * v0
    for prec, tol in (("f64", 2e-3), ("f32", 3e-3)):
        en, mom, deepest, vs = runs[prec]
        assert np.abs(en / e0 - 1.0).max() < tol, (prec, np.abs(en / e0 - 1.0).max())      # bounded O(dt^2) oscillation of the Verlet scheme
        assert np.abs(mom).max() < (1e-12 if prec == "f64" else 1e-5) * m * v0
        assert abs(vs[1, 0] - vs[0, 0]) / (2 * v0) > 0.995                                  # they part with the speeds they came with
    assert np.abs(runs["f32"][0] - runs["f64"][0]).max() < 1e-3 * e0                        # the fp32 curve lies on the fp64 one
    assert abs(runs["f32"][2] / runs["f64"][2] - 1.0) < 1e-3
    dmax = (15.0 * (m / 2) * (2 * v0) ** 2 / (16.0 * Ystar * np.sqrt(Rstar))) ** 0.4         # Hertz impact, closed form
    assert abs(runs["f64"][2] / dmax - 1.0) < 5e-3


def test_f32_and_f64_handles_do_not_mix():
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Dem
    pd, x, v, w, R = W.dem_random(5, 200, box=(5.0, 5.0, 5.0))
    g32, g64 = Dem(pd, x, v, w, R, precision="f32"), Dem(pd, x, v, w, R)
    with pytest.raises(L.LeddsError):
        L.ledds_dem_step(g32.h, g64.x, g64.v, g64.w, g64.a, g64.alpha, g64.radius, None, None, g32.history, g32.scratch, g32.status, 1)
    with pytest.raises(L.LeddsError):
        L.ledds_dem_step_f32(g64.h, g32.x, g32.v, g32.w, g32.a, g32.alpha, g32.radius, None, None, g64.history, g64.scratch, g64.status, 1)
    sb32, hb32 = L.ledds_dem_workspace_bytes_f32(g32.p)
    sb64, hb64 = L.ledds_dem_workspace_bytes(g64.p)
    assert hb32 < 0.6 * hb64 and sb32 < sb64


def test_f32_full_size_config5_dense_ordering_and_contacts():
    # BASELINE configs[4] size in single precision, the launch configuration bench.py times: the ordering is the stable
    # argsort of the fp32 keys, the contact count is that of the fp64 run up to the contacts within rounding of delta_n = 0
    pd, x, v, w, R = W.cfg5_pour(dense=True)
    from paper_2512_04997_b200 import Dem
    g = Dem(pd, x, v, w, R, precision="f32")
    q = g.query(pair_cap=8_000_000)
    key = keys32(pd, g.state()["x"])
    idx = np.argsort(key, kind="stable").astype(np.uint32)
    assert np.array_equal(q["idx"], idx) and q["status"] == 0
    g64 = Dem(pd, x, v, w, R)
    n64 = len(g64.query(pair_cap=8_000_000)["pairs"])
    assert abs(len(q["pairs"]) - n64) <= 2e-3 * n64
