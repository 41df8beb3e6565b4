"""GPU parity: coupled PSM step (ledds_coupled_step) vs the CPU oracle."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


PATHS = {"one_launch": {}, "chain_radix": {"no_single_block": 1, "cell_order": 1},
         "chain_counting": {"no_single_block": 1, "cell_order": 2}}


@pytest.fixture(params=list(PATHS))
def dem_path(request):
    """The tests that name this fixture run on every path of the step: small systems (n <= 4 096) by the single-launch cluster
    kernel, and the chain of kernels that larger systems take with the order by cell from the radix passes and from
    the counting sort (ledds_dem_params.no_single_block, cell_order)."""
    from paper_2512_04997_b200 import Dem
    old = Dem.DEFAULTS
    Dem.DEFAULTS = PATHS[request.param]
    yield request.param
    Dem.DEFAULTS = old


def both(lbm, cpl, pd, x, v, w, R, u=None):
    import oracle
    from paper_2512_04997_b200 import Coupled, Dem, Lbm
    f0 = oracle.lbm_equilibrium(lbm["shape"], None, u)
    od = oracle.Dem(pd, x, v, w, R)
    o = oracle.Coupled(lbm, cpl, od, f0)
    gl = Lbm(lbm, None, u)
    gd = Dem(pd, x, v, w, R)
    g = Coupled(gl, gd, cpl, float(np.max(R)))
    return o, g


ACHIEVED = {}          # test name -> largest errors seen (printed by pytest -s; quoted in DESIGN.md section 11)


def compare(o, g, tol_f=1e-12, tol_F=1e-10, name=None):
    """Populations 1e-12 of max |f|.  Forces: the momentum exchange of Eq. 41 is a sum of differences
    of O(1) populations, so its rounding floor is ~1e-17 per term whatever the size of the force:
    tolerance = tol_F * max|F| + FLOOR, FLOOR = 1e-13 lattice units converted to the units the problem is posed
    in (rho_f dx^4 / Dt^2 for a force, one more dx for a torque, dx / Dt for a velocity, 1 / Dt for a spin)."""
    dx, rho_f = o.cpl["dx"], o.cpl["rho_f"]
    Dt = o.cpl["n_sub"] * o.dem.p.dt
    FLOOR = 1e-13
    fF, fM = FLOOR * rho_f * dx ** 4 / Dt ** 2, FLOOR * rho_f * dx ** 5 / Dt ** 2
    f = g.lbm.export()
    ef = np.abs(f - o.f).max() / np.abs(o.f).max()
    assert ef <= tol_f
    F, M = g.f_hyd.cpu().numpy(), g.m_hyd.cpu().numpy()
    Rm = float(o.dem.R.max()) / dx
    eF = np.abs(F - o.F_sf).max() / max(np.abs(o.F_sf).max(), 1e-300)
    assert np.abs(F - o.F_sf).max() <= tol_F * np.abs(o.F_sf).max() + fF
    assert np.abs(M - o.M_sf).max() <= tol_F * np.abs(o.M_sf).max() + fM * Rm
    s = g.dem.state()
    L = max(o.lbm["shape"]) * dx
    ex = np.abs(s["x"] - o.dem.x).max() / L
    assert ex <= 1e-9
    assert np.abs(s["v"] - o.dem.v).max() <= 1e-9 * np.abs(o.dem.v).max() + FLOOR * dx / Dt
    assert np.abs(s["w"] - o.dem.w).max() <= 1e-9 * np.abs(o.dem.w).max() + FLOOR / Dt
    assert int(g.dem.status[0].item()) == o.status
    if name:
        ACHIEVED[name] = (ef, eF, ex)
        print(f"{name}: |df|/|f| = {ef:.1e}  |dF|/|F| = {eF:.1e}  |dx|/L = {ex:.1e}")


def test_single_sphere_settling_small():
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 64), R=5.0, z0=40.0, g=1e-3)
    o, g = both(lbm, cpl, pd, x, v, w, R)
    o.step(1); g.step(1)
    compare(o, g)
    o.step(9); g.step(9)
    compare(o, g)
    assert o.F_sf[0, 2] > 0 and o.dem.v[0, 2] < 0


def test_zero_reach_particle_is_plain_lbm_bit_exact():
    # no solid in any cell -> the coupled kernel is the plain stream-collide, bit for bit
    from paper_2512_04997_b200 import Lbm
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(64, 16, 16), R=3.0, z0=8.0, g=0.0)
    pd = dict(pd); pd["lo"] = (-0.5, -0.5, -100.5); pd["bc"] = (1, 1, 1)
    x = np.array([[8.0, 8.0, -50.0]])                          # far below the lattice
    lbm = dict(lbm); cpl = dict(cpl)
    rho, u = W.random_flow(lbm["shape"], 4)
    import oracle
    from paper_2512_04997_b200 import Coupled, Dem
    gl = Lbm(dict(lbm, variant=1), rho, u)
    gd = Dem(pd, x, v, w, R)
    g = Coupled(gl, gd, cpl, 3.0)
    g.step(5)
    plain = Lbm(dict(lbm, variant=1), rho, u)
    plain.step(5)
    assert np.array_equal(gl.export(), plain.export())
    assert np.all(g.f_hyd.cpu().numpy() == 0)


@pytest.mark.usefixtures("dem_path")
def test_shear_suspension_small_with_contacts_and_periodic_wrap():
    # config-4 shaped: periodic x,y, moving z walls, spheres placed by RSA, some across the periodic seam
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=2, n=64, n_part=60, R=4.0)
    x[0] = (0.2, 30.0, 20.0); x[1] = (63.3, 10.0, 40.0)          # straddle the x seam (kept apart from others below)
    keep = np.ones(len(x), bool)
    for i in (0, 1):
        d = x - x[i]; d[:, :2] -= 64 * np.round(d[:, :2] / 64)
        close = (np.linalg.norm(d, axis=1) < 2 * 4.0); close[i] = False
        keep &= ~close
    x, v, w, R = x[keep], v[keep], w[keep], R[keep]
    pd = dict(pd); pd["n"] = len(x)
    # give two spheres an overlap so the DEM contact path is active inside the coupled step
    x[3] = x[2] + np.array([7.5, 0.0, 0.0]); x[3, 0] %= 64
    o, g = both(lbm, cpl, pd, x, v, w, R, u)
    o.step(1); g.step(1)
    compare(o, g)
    o.step(4); g.step(4)
    compare(o, g)
    assert np.abs(o.F_sf).max() > 0


@pytest.mark.usefixtures("dem_path")
def test_substepping():
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 48), R=4.0, z0=5.0, g=2e-3)
    cpl = dict(cpl, n_sub=4); pd = dict(pd, dt=0.25)
    o, g = both(lbm, cpl, pd, x, v, w, R)
    o.step(6); g.step(6)
    compare(o, g)


def test_three_solids_in_a_cell_are_flagged():
    import paper_2512_04997_b200 as L
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 32), R=3.0, z0=16.0, g=0.0)
    pd = dict(pd, n=3, kn=1e-9, kn_w=1e-9, kt=1e-9, kt_w=1e-9)
    x = np.array([[15.0, 16.0, 16.0], [17.0, 16.0, 16.0], [16.0, 17.5, 16.0]])
    z = np.zeros((3, 3))
    o, g = both(lbm, cpl, pd, x, z, z, np.full(3, 3.0))
    o.step(1); g.step(1)
    assert o.status & 2 and int(g.dem.status[0].item()) & L.ST_SOLID_OVERFLOW
    compare(o, g)


def test_ragged_row_and_64bit_index_path():
    # nx = 72: the last 128-wide block of a row is mostly past the row end; variant 3 forces the 64-bit
    # index instantiation that lattices with 19 N >= 2^32 take
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=3, n=72, n_part=40, R=4.0)
    for variant in (0, 3):
        o, g = both(dict(lbm, variant=variant), cpl, pd, x, v, w, R, u)
        o.step(3); g.step(3)
        compare(o, g)


def test_two_solid_cells_take_the_second_solid():
    # two spheres whose shells (R + r_c) overlap without touching: cells cut by both must carry both weights
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(48, 32, 32), R=4.0, z0=16.0, g=0.0)
    pd = dict(pd, n=2)
    x = np.array([[19.6, 16.2, 16.0], [28.3, 15.7, 16.4]])            # gap 0.7 < 2 r_c
    vv = np.array([[0.01, 0.0, 0.0], [-0.01, 0.005, 0.0]]); ww = np.array([[0, 0, 0.002], [0.001, 0, 0]])
    o, g = both(lbm, cpl, pd, x, vv, ww, np.full(2, 4.0))
    o.step(2); g.step(2)
    compare(o, g)
    assert o.status == 0


def test_full_size_config3_one_step():
    # BASELINE configs[3] at full size in the launch configuration bench.py times: one coupled step against
    # the oracle (all forces; populations on every 7th cell)
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear()
    o, g = both(lbm, cpl, pd, x, v, w, R, u)
    o.step(1); g.step(1)
    F, M = g.f_hyd.cpu().numpy(), g.m_hyd.cpu().numpy()
    assert np.abs(F - o.F_sf).max() <= 1e-10 * np.abs(o.F_sf).max() + 1e-13
    assert np.abs(M - o.M_sf).max() <= 1e-10 * np.abs(o.M_sf).max() + 4e-13
    s = g.dem.state()
    assert np.abs(s["x"] - o.dem.x).max() <= 1e-9 * 256
    assert int(g.dem.status[0].item()) == o.status == 0
    f = g.lbm.export()
    assert np.abs(f[:, ::7] - o.f[:, ::7]).max() <= 1e-12 * np.abs(o.f).max()


def test_empty_particle_system_is_plain_lbm():
    # n = 0 is a valid input: the coupled step is then the plain stream-collide, bit for bit, and DEM calls are no-ops
    import oracle
    from paper_2512_04997_b200 import Coupled, Dem, Lbm
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(48, 12, 10), R=3.0, z0=5.0, g=0.0)
    pd = dict(pd, n=0)
    e3, e1 = np.zeros((0, 3)), np.zeros(0)
    rho, u = W.random_flow(lbm["shape"], 9)
    gl = Lbm(dict(lbm, variant=1), rho, u)
    gd = Dem(pd, e3, e3, e3, e1)
    g = Coupled(gl, gd, cpl, 3.0)
    g.step(4)
    gd.step(3)
    q = gd.query()
    assert len(q["pairs"]) == 0 and q["status"] == 0
    plain = Lbm(dict(lbm, variant=1), rho, u)
    plain.step(4)
    assert np.array_equal(gl.export(), plain.export())
    ref = oracle.lbm_run(lbm["shape"], oracle.lbm_equilibrium(lbm["shape"], rho, u), lbm["tau"], 4, bc=lbm["bc"])
    assert np.abs(gl.export() - ref).max() <= 1e-13 * np.abs(ref).max()


def test_hydrodynamic_force_is_bit_reproducible():
    # the per-solid sums are exact integer sums: two runs of the same problem agree bit for bit
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=5, n=64, n_part=120, R=4.0)
    out = []
    for _ in range(2):
        o, g = both(lbm, cpl, pd, x, v, w, R, u)
        g.step(6)
        out.append((g.f_hyd.cpu().numpy().copy(), g.m_hyd.cpu().numpy().copy(), g.lbm.export()))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert np.array_equal(out[0][2], out[1][2])


def test_trt_coupled_step():
    # Eq. (33) with the TRT operator of Eq. (30) as Omega_i (the model of the paper's results), moving walls,
    # contacts, two-solid cells
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=7, n=64, n_part=90, R=4.0)
    o, g = both(dict(lbm, collision=1), cpl, pd, x, v, w, R, u)
    o.step(1); g.step(1)
    compare(o, g)
    o.step(5); g.step(5)
    compare(o, g)


@pytest.mark.parametrize("collision", [0, 1])
def test_subdivision_solid_fraction(collision):
    # Eq. (38), 10^3 points per cell (the paper's validation setting), with BGK and with TRT: the counts are
    # integers, so the weights must agree exactly and the step to the usual tolerances
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=8, n=64, n_part=70, R=4.0)
    cpl = dict(cpl, solid_fraction=1)
    o, g = both(dict(lbm, collision=collision), cpl, pd, x, v, w, R, u)
    o.step(1); g.step(1)
    compare(o, g)
    o.step(3); g.step(3)
    compare(o, g)
    assert np.abs(o.F_sf).max() > 0


def test_subdivision_single_sphere_walls():
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 48), R=5.3, z0=30.0, g=1e-3)
    o, g = both(lbm, dict(cpl, solid_fraction=1), pd, x, v, w, R)
    o.step(6); g.step(6)
    compare(o, g)


def test_paper_bed_workload_small():
    # SURVEY 8(f) rank 3 in small: the generator of the paper's performance workload (TRT, 10 DEM sub-steps per
    # LBM step, periodic x y, walls z) on a 96 x 48 x 64 lattice with spheres of 12 cells diameter at phi = 0.3
    lbm, cpl, pd, x, v, w, R = W.paper_bed(0.30, shape=(96, 48, 64), D=12.0)
    assert len(R) > 30
    o, g = both(lbm, cpl, pd, x, v, w, R)
    o.step(2); g.step(2)
    compare(o, g)


def posed_in_units(L, T, rho_f, origin, n_sub):
    """The two-sphere settling problem of tests/test_oracle_coupled.py, posed in units of length L, time T, mass
    rho_f L^3 with the lattice origin at `origin` of the DEM frame (the oracle's conversions are pinned there)."""
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(40, 24, 40), R=3.6, z0=22.0, g=2e-3)
    x = np.array([[11.0, 10.0, 22.0], [15.3, 11.0, 26.3]]); R = np.array([3.6, 2.9])
    v = np.tile(np.array([[0.004, -0.002, 0.0]]), (2, 1)); w = np.tile(np.array([[0.001, 0.002, -0.0015]]), (2, 1))
    Mu = rho_f * L ** 3
    org = np.asarray(origin, float)
    pdB = dict(pd, n=2)
    pdB.update(lo=tuple(org + L * np.asarray(pd["lo"])), hi=tuple(org + L * np.asarray(pd["hi"])), cell=pd["cell"] * L,
               dt=T / n_sub, g=tuple(np.asarray(pd["g"]) * L / T ** 2), density=pd["density"] * Mu / L ** 3)
    for k in ("kn", "kt", "kn_w", "kt_w"):
        pdB[k] = pd[k] * Mu / T ** 2
    cplB = dict(n_sub=n_sub, dx=L, rho_f=rho_f, origin=tuple(org))
    return lbm, cplB, pdB, org + L * x, v * L / T, w / T, R * L


@pytest.mark.usefixtures("dem_path")
@pytest.mark.parametrize("n_sub", [1, 4])
@pytest.mark.parametrize("units", [(0.5, 0.25, 2.0, (3.0, -1.5, 0.25)), (3.0e-4, 7.0e-4, 998.2, (0.0123, -0.4, 1.7))])
def test_units_and_origin_of_the_coupling(units, n_sub):
    # ledds_cpl_params.dx, rho_f, origin and n_sub * dt != 1 (reading G32): x_k = (x - origin)/dx, v_k Dt/dx, w_k Dt,
    # force scale rho_f dx^4/Dt^2, torque scale rho_f dx^5/Dt^2 on the CUDA path against the oracle
    Lu, T, rho_f, org = units
    lbm, cpl, pd, x, v, w, R = posed_in_units(Lu, T, rho_f, org, n_sub)
    o, g = both(lbm, cpl, pd, x, v, w, R)
    o.step(1); g.step(1)
    compare(o, g)
    o.step(9); g.step(9)
    compare(o, g, name=f"units dx={Lu} n_sub={n_sub}")
    assert np.abs(o.F_sf).max() > 1e-4 * rho_f * Lu ** 4 / T ** 2


def test_radius_above_r_max_is_flagged():
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Coupled, Dem, Lbm
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 32), R=4.0, z0=16.0, g=0.0)
    g = Coupled(Lbm(lbm), Dem(pd, x, v, w, R), cpl, 3.5)       # the caller promised r_max = 3.5
    g.step(1)
    assert int(g.dem.status[0].item()) & L.ST_RADIUS_RANGE
    g = Coupled(Lbm(lbm), Dem(pd, x, v, w, R), cpl, 4.0)
    g.step(1)
    assert int(g.dem.status[0].item()) == 0


def test_full_size_config2_settling_20_steps():
    # BASELINE configs[2] at full size (64 x 64 x 256, walls on all sides, tau = 0.55, one sphere R = 6, density ratio
    # 1.5): 20 coupled steps in the launch configuration bench.py times (the BX = 64 instantiation), all populations
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling()
    o, g = both(lbm, cpl, pd, x, v, w, R)
    o.step(20); g.step(20)
    compare(o, g, name="configs[2] full size, 20 steps")
    assert o.dem.v[0, 2] < 0 and o.F_sf[0, 2] > 0


@pytest.mark.usefixtures("dem_path")
def test_coupled_100_steps_small():
    # drift between the two implementations shows late: 100 coupled steps of a sheared suspension with contacts,
    # two-solid cells and periodic wrap
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=11, n=48, n_part=40, R=4.0)
    o, g = both(lbm, cpl, pd, x, v, w, R, u)
    for _ in range(4):
        o.step(25); g.step(25)
        compare(o, g, name="48^3 shear, 100 steps")


# ------------------------------------------------------------------------------------ fp32 lattice
# ledds_coupled_step_f32: populations, moments and collision in fp32; solid geometry, force sums and DEM in fp64.
# Bounds: populations as for the plain fp32 lattice, 8 * steps * 2^-24 * max|f|.  A cell's
# term of Eq. (41) is B rho (u - u_k) with rho u = sum_i c_i f_i, ten populations per axis, so a solid's force
# differs from the fp64 one by at most (cells it cuts) * 10 * that bound per component, and its torque by
# (R + r_c + 1) times as much; the observed differences are far smaller (the errors of the cells do not add up
# coherently), and the test also asserts them against 1e-3 of the largest force.
EPS32 = 2.0 ** -24


def both_f32(lbm, cpl, pd, x, v, w, R, u=None):
    import oracle
    from paper_2512_04997_b200 import Coupled, Dem, Lbm
    u32 = None if u is None else u.astype(np.float32)
    f0 = oracle.lbm_equilibrium(lbm["shape"], None, None if u is None else u32.astype(np.float64))
    o = oracle.Coupled(lbm, cpl, oracle.Dem(pd, x, v, w, R), f0)
    g = Coupled(Lbm(lbm, None, u32, precision="f32"), Dem(pd, x, v, w, R), cpl, float(np.max(R)))
    return o, g


def compare_f32(o, g, steps, cpl):
    f = g.lbm.export().astype(np.float64)
    pop = 8 * steps * EPS32 * np.abs(o.f).max()
    assert np.abs(f - o.f).max() <= pop
    Rm = float(o.dem.R.max())
    reach = Rm / cpl["dx"] + 1.0
    cells = (2 * reach + 1) ** 3
    F, M = g.f_hyd.cpu().numpy(), g.m_hyd.cpu().numpy()
    # lattice units -> DEM units: force rho_f dx^4 / Dt^2, torque one more dx (set-ups here have all three = 1)
    dF, dM = np.abs(F - o.F_sf).max(), np.abs(M - o.M_sf).max()
    assert dF <= cells * 10 * pop and dM <= cells * 10 * pop * (reach + 1)
    assert dF <= 1e-3 * np.abs(o.F_sf).max() + 1e-7 and dM <= 1e-3 * np.abs(o.M_sf).max() + 1e-7 * Rm
    s = g.dem.state()
    assert np.abs(s["x"] - o.dem.x).max() <= 1e-5 * max(o.lbm["shape"])
    assert int(g.dem.status[0].item()) == o.status
    return dF / (np.abs(o.F_sf).max() + 1e-300), np.abs(f - o.f).max() / np.abs(o.f).max()


@pytest.mark.parametrize("collision", [0, 1])
def test_f32_single_sphere_settling(collision):
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 64), R=5.0, z0=40.0, g=1e-3)
    lbm = dict(lbm, collision=collision)
    o, g = both_f32(lbm, cpl, pd, x, v, w, R)
    o.step(10); g.step(10)
    compare_f32(o, g, 10, cpl)


def test_f32_shear_suspension_with_two_solid_cells_and_wrap():
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=2, n=64, n_part=60, R=4.0)
    o, g = both_f32(lbm, cpl, pd, x, v, w, R, u)
    o.step(5); g.step(5)
    compare_f32(o, g, 5, cpl)


def test_f32_ragged_64bit_and_subdivision():
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=3, n=72, n_part=40, R=4.0)
    lbm = dict(lbm, variant=3, collision=1)
    cpl = dict(cpl, solid_fraction=1)
    o, g = both_f32(lbm, cpl, pd, x, v, w, R, u)
    o.step(3); g.step(3)
    compare_f32(o, g, 3, cpl)


def test_f32_handle_is_rejected_by_the_fp64_call():
    import paper_2512_04997_b200 as L
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(32, 32, 32), R=3.0, z0=16.0, g=0.0)
    o, g = both_f32(lbm, cpl, pd, x, v, w, R)
    d = g.dem
    with pytest.raises(L.LeddsError):
        L.ledds_coupled_step(g.lbm.h, d.h, g.c, g.r_max, g.lbm.f, d.x, d.v, d.w, d.a, d.alpha, d.radius, g.f_hyd, g.m_hyd,
                             d.history, d.scratch, g.cpl_scratch, d.status, 1)


def test_f32_full_size_config3_one_step():
    # the configuration bench.py times as sub.cfg4_f32_lattice: 256^3, 20 000 spheres, one coupled step
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear()
    o, g = both_f32(lbm, cpl, pd, x, v, w, R, u)
    o.step(1); g.step(1)
    compare_f32(o, g, 1, cpl)
