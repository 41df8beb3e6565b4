"""GPU parity: CUDA stream-collide (through the C ABI) vs the CPU oracle, element by element
(north_star: populations after 100 steps within 1e-12 of max |f|)."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-12


def run_pair(shape, tau, bc, u_wall, steps, variant, seed=0, flow="random", collision=0):
    import oracle
    from paper_2512_04997_b200 import Lbm
    rho, u = W.random_flow(shape, seed) if flow == "random" else W.tgv(shape, 0.02, 1.0, "xy")
    lbm = dict(shape=shape, tau=tau, bc=bc, u_wall=u_wall, variant=variant, collision=collision)
    g = Lbm(lbm, rho, u)
    f0 = g.export()
    ref0 = oracle.lbm_equilibrium(shape, rho, u)
    assert np.abs(f0 - ref0).max() <= 1e-15                    # init (Eq. 28) agrees
    g.step(steps)
    f = g.export()
    ref = oracle.lbm_run(shape, ref0, tau, steps, bc=bc, u_wall=u_wall, trt=bool(collision))
    return f, ref


MOVING = np.zeros((3, 2, 3))
MOVING[2, 0, 0] = -0.05; MOVING[2, 1, 0] = 0.05; MOVING[1, 0, 2] = 0.02; MOVING[0, 1, 1] = -0.03


@pytest.mark.parametrize("variant", [1, 3])
@pytest.mark.parametrize("shape,bc,uw", [
    ((64, 12, 10), (0, 0, 0), None),
    ((64, 12, 10), (1, 1, 1), MOVING),
    ((128, 6, 5), (0, 0, 1), MOVING),
    ((64, 7, 9), (1, 0, 0), MOVING),
    ((64, 8, 8), (0, 1, 0), None),
])
def test_populations_after_100_steps(variant, shape, bc, uw):
    f, ref = run_pair(shape, 0.6, bc, uw, 100, variant)
    assert np.abs(f - ref).max() <= TOL * np.abs(ref).max()


@pytest.mark.parametrize("variant", [1, 3])
@pytest.mark.parametrize("shape,bc,uw", [((64, 12, 10), (0, 0, 0), None), ((64, 9, 10), (1, 0, 1), MOVING), ((37, 6, 5), (0, 1, 0), MOVING)])
def test_trt_populations_after_100_steps(variant, shape, bc, uw):
    # PAPER.md:236-246, Eq. (29)-(31): the collision model the paper's results use
    f, ref = run_pair(shape, 0.56, bc, uw, 100, variant, collision=1)
    assert np.abs(f - ref).max() <= TOL * np.abs(ref).max()


@pytest.mark.parametrize("shape", [(37, 5, 3), (1, 1, 1), (130, 3, 2), (5, 1, 7)])
def test_ragged_sizes(shape):
    # nx not a multiple of the block width; single cells and thin boxes work
    f, ref = run_pair(shape, 0.8, (0, 1, 0), MOVING, 20, 0)
    assert np.abs(f - ref).max() <= TOL * np.abs(ref).max()


def test_index_widths_agree_bit_for_bit():
    # the 32-bit and the 64-bit index instantiations are the same arithmetic: equal bit for bit after 10 steps
    import paper_2512_04997_b200  # noqa
    f1, _ = run_pair((64, 8, 8), 0.7, (1, 0, 1), MOVING, 10, 1)
    f2, _ = run_pair((64, 8, 8), 0.7, (1, 0, 1), MOVING, 10, 3)
    assert np.array_equal(f1, f2)


def test_mass_conserved_and_tgv_decay_config2_small():
    import oracle
    from paper_2512_04997_b200 import Lbm
    shape = (64, 64, 64)
    rho, u = W.tgv(shape, 0.02, 1.0, "xy")
    g = Lbm(dict(shape=shape, tau=0.6, bc=(0, 0, 0), u_wall=None), rho, u)
    f0 = g.export()
    g.step(100); _, r1, u1 = g.export(want_moments=True)
    g.step(400); f2, r2, u2 = g.export(want_moments=True)
    assert abs(f2.sum() - f0.sum()) <= 1e-12 * f0.sum()
    rate = 4.0 * (0.1 / 3.0) * (2 * np.pi / 64) ** 2
    assert abs(np.log((u1 ** 2).sum() / (u2 ** 2).sum()) / 400 / rate - 1.0) < 0.005


def test_full_size_config2_100_steps_against_oracle():
    # north_star: "lattice populations after 100 steps within 1e-12" at BASELINE configs[1] itself: 128^3 periodic
    # Taylor-Green field, tau = 0.6, the launch configuration bench.py times; every population of every cell
    import oracle
    from paper_2512_04997_b200 import Lbm
    lbm, rho, u = W.cfg2_tgv(128)
    g = Lbm(lbm, rho, u)
    g.step(100)
    f = g.export()
    ref = oracle.lbm_run(lbm["shape"], oracle.lbm_equilibrium(lbm["shape"], rho, u), lbm["tau"], 100)
    err = np.abs(f - ref).max() / np.abs(ref).max()
    print(f"configs[1] 128^3 x 100 steps: max |df| / max |f| = {err:.2e}")
    assert err <= TOL


TWO_AXES = np.zeros((3, 2, 3))
TWO_AXES[1, 0] = (0.01, 0.0, 0.03); TWO_AXES[1, 1] = (-0.02, 0.0, -0.04)     # y walls slide along x and z
TWO_AXES[2, 0] = (0.02, -0.05, 0.0); TWO_AXES[2, 1] = (0.0, 0.035, 0.0)      # z walls slide along x and y


@pytest.mark.parametrize("collision", [0, 1])
@pytest.mark.parametrize("shape,bc", [((64, 6, 5), (0, 1, 1)), ((37, 7, 6), (1, 1, 1))])
def test_corner_links_crossing_two_moving_walls(shape, bc, collision):
    # reading G19: a link that leaves through two walls takes the sum of c_i.u_w over both (pinned for the oracle by
    # exact mass conservation, tests/test_oracle_lbm.py); here every edge and corner of the box has moving walls
    uw = TWO_AXES.copy()
    if bc[0]:
        uw[0, 0] = (0.0, 0.02, -0.01); uw[0, 1] = (0.0, -0.03, 0.015)
    f, ref = run_pair(shape, 0.7, bc, uw, 100, 1, seed=3, collision=collision)
    assert np.abs(f - ref).max() <= TOL * np.abs(ref).max()


def test_import_roundtrip_and_errors():
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Lbm
    shape = (64, 4, 4)
    f0 = np.random.default_rng(0).random((19, 64 * 16)) + 0.5
    g = Lbm(dict(shape=shape, tau=0.9, bc=(0, 0, 0), u_wall=None), f_canonical=f0)
    assert np.array_equal(g.export(), f0)
    with pytest.raises(L.LeddsError):
        Lbm(dict(shape=(37, 4, 4), tau=0.9, bc=(0, 0, 0), u_wall=None, variant=2))      # no such kernel
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_step(g.h, g.f[1:], 1)                    # misaligned pointer -> LEDDS_EALIGN


# ------------------------------------------------------------------------------------ fp32 variant
# the paper's single-precision runs.  The oracle stays fp64; the bound on the difference
# is the rounding of the fp32 arithmetic: every step adds at most ~8 roundings of size
# 2^-24 max|f| to a population (tree sums of Eq. 22, Eq. 28, Eq. 26), so after `steps` steps
# |f32 - f64| <= 8 * steps * 2^-24 * max|f|; the observed difference is ~sqrt(steps) of that.
EPS32 = 2.0 ** -24


def run_pair_f32(shape, tau, bc, u_wall, steps, variant, collision=0, seed=0):
    import oracle
    from paper_2512_04997_b200 import Lbm
    rho, u = W.random_flow(shape, seed)
    rho, u = rho.astype(np.float32), u.astype(np.float32)     # both sides start from the same fp32 fields
    lbm = dict(shape=shape, tau=tau, bc=bc, u_wall=u_wall, variant=variant, collision=collision)
    g = Lbm(lbm, rho, u, precision="f32")
    f0 = g.export()
    assert f0.dtype == np.float32
    ref0 = oracle.lbm_equilibrium(shape, rho.astype(np.float64), u.astype(np.float64))
    assert np.abs(f0 - ref0).max() <= 4 * EPS32 * np.abs(ref0).max()
    g.step(steps)
    f = g.export()
    ref = oracle.lbm_run(shape, ref0, tau, steps, bc=bc, u_wall=u_wall, trt=bool(collision))
    return f.astype(np.float64), ref


@pytest.mark.parametrize("variant,collision", [(1, 0), (3, 0), (1, 1)])
@pytest.mark.parametrize("shape,bc,uw", [
    ((64, 12, 10), (0, 0, 0), None),
    ((64, 12, 10), (1, 1, 1), MOVING),
    ((130, 6, 5), (0, 0, 1), MOVING),
    ((37, 7, 9), (1, 0, 0), MOVING),
])
def test_f32_populations_after_100_steps(variant, collision, shape, bc, uw):
    f, ref = run_pair_f32(shape, 0.6, bc, uw, 100, variant, collision)
    err = np.abs(f - ref).max() / np.abs(ref).max()
    assert err <= 8 * 100 * EPS32
    assert np.sqrt(np.mean((f - ref) ** 2)) <= 8 * 10 * EPS32 * np.abs(ref).max()    # random-walk growth


def test_f32_tgv_decay_and_mass():
    from paper_2512_04997_b200 import Lbm
    shape = (64, 64, 64)
    rho, u = W.tgv(shape, 0.02, 1.0, "xy")
    g = Lbm(dict(shape=shape, tau=0.6, bc=(0, 0, 0), u_wall=None), rho, u, precision="f32")
    f0 = g.export().astype(np.float64)
    g.step(100); _, r1, u1 = g.export(want_moments=True)
    g.step(400); f2, r2, u2 = g.export(want_moments=True)
    assert abs(f2.astype(np.float64).sum() - f0.sum()) <= 500 * EPS32 * f0.sum()
    rate = 4.0 * (0.1 / 3.0) * (2 * np.pi / 64) ** 2
    e1, e2 = (u1.astype(np.float64) ** 2).sum(), (u2.astype(np.float64) ** 2).sum()
    assert abs(np.log(e1 / e2) / 400 / rate - 1.0) < 0.01


def test_f32_full_size_config2_against_oracle():
    import oracle
    from paper_2512_04997_b200 import Lbm
    lbm, rho, u = W.cfg2_tgv(128)
    rho, u = rho.astype(np.float32), u.astype(np.float32)
    g = Lbm(lbm, rho, u, precision="f32")
    g.step(10)
    f = g.export().astype(np.float64)
    ref = oracle.lbm_run(lbm["shape"], oracle.lbm_equilibrium(lbm["shape"], rho.astype(np.float64), u.astype(np.float64)),
                         lbm["tau"], 10)
    assert np.abs(f - ref).max() <= 8 * 10 * EPS32 * np.abs(ref).max()


def test_f32_handles_and_fp64_calls_do_not_mix():
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Lbm
    lbm = dict(shape=(64, 4, 4), tau=0.9, bc=(0, 0, 0), u_wall=None)
    g32, g64 = Lbm(lbm, precision="f32"), Lbm(lbm)
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_step(g32.h, g64.f, 1)
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_step_f32(g64.h, g32.f, 1)
    with pytest.raises(L.LeddsError):
        Lbm(dict(lbm, variant=2), precision="f32")           # no such kernel
    f0 = (np.random.default_rng(1).random((19, 64 * 16)) + 0.5).astype(np.float32)
    g = Lbm(lbm, f_canonical=f0, precision="f32")
    assert np.array_equal(g.export(), f0)
