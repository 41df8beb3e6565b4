"""Pins for oracle/psm.c (SURVEY 8(c.5) xii-xvi; readings G21-G26).  CPU only."""
import numpy as np
import pytest

import oracle
import workloads as W


def momentum(f):
    cx, cy, cz, opp, t = oracle.lattice()
    return f.sum(1) @ np.stack([cx, cy, cz], 1).astype(float)


def test_weights_B_limits():
    # Eq. 36: B(0) = 0, B(1) = 1, monotone; Eq. 39: beta clamps to [0, 1]
    for tau in (0.55, 0.6, 1.0):
        assert oracle.psm_B(0.0, tau) == 0.0 and abs(oracle.psm_B(1.0, tau) - 1.0) < 1e-15
        b = [oracle.psm_B(x, tau) for x in np.linspace(0, 1, 11)]
        assert np.all(np.diff(b) > 0)
    assert abs(oracle.psm_B(0.5, 1.0) - 0.25 / 1.0) < 1e-15          # 0.5*0.5/(0.5+0.5)
    rc = oracle.psm_rc()
    assert abs(4 / 3 * np.pi * rc ** 3 - 1.0) < 1e-14                 # Eq. 40: sphere of volume dx^3
    assert oracle.psm_beta(4.0, 4.0 + rc) == 0.0 and abs(oracle.psm_beta(4.0, 4.0 - rc) - 1.0) < 1e-15
    assert abs(oracle.psm_beta(4.0, 4.0) - 0.5) < 1e-15 and oracle.psm_beta(4.0, 0.0) == 1.0


def test_sum_of_beta_is_the_sphere_volume():
    # G25: distance-based fraction integrates to 4/3 pi R^3 within a few per cent
    for R, xk in ((4.0, (10.3, 11.1, 9.7)), (6.0, (12.0, 12.5, 11.9))):
        s = oracle.psm_beta_sum((24, 24, 24), (1, 1, 1), np.array(xk), R)
        assert abs(s / (4 / 3 * np.pi * R ** 3) - 1.0) < 0.03


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1)])
def test_no_particle_is_plain_lbm_bit_for_bit(bc):
    # PAPER.md:297 "reverts to the standard Collide and Stream"
    shape = (7, 6, 5)
    rho, u = W.random_flow(shape, 1)
    f = oracle.lbm_equilibrium(shape, rho, u)
    uw = np.zeros((3, 2, 3)); uw[2, 1, 0] = 0.03
    a = oracle.lbm_run(shape, f, 0.7, 1, bc=bc, u_wall=uw)
    b, F, M, st = oracle.psm_step(shape, f, 0.7, bc, uw, np.zeros((0, 3)), np.zeros((0, 3)), np.zeros((0, 3)), np.zeros(0))
    assert np.array_equal(a, b) and st == 0
    # a sphere far outside reach of every node changes nothing either
    b2, F, M, st = oracle.psm_step(shape, f, 0.7, (1, 1, 1), uw, [[-50.0, 3, 3]], [[0.1, 0, 0]], [[0, 0, 0]], [2.0])
    a2 = oracle.lbm_run(shape, f, 0.7, 1, bc=(1, 1, 1), u_wall=uw)
    assert np.array_equal(a2, b2) and np.all(F == 0)


@pytest.mark.parametrize("trt", [False, True])
def test_momentum_budget_periodic(trt):
    # G26: in a periodic box the fluid momentum changes by exactly minus the force on the solids
    # (lattice units): sum f' c - sum f c = - sum_k F_k.  Also mass is conserved (sum_i Omega^s = 0).
    shape = (16, 14, 12)
    rho, u = W.random_flow(shape, 2, amp=0.01)
    f = oracle.lbm_equilibrium(shape, rho, u)
    xk = np.array([[5.2, 6.1, 5.7], [11.3, 6.4, 6.2], [15.6, 1.0, 11.5]])      # third wraps around
    vk = np.array([[0.02, 0.0, -0.01], [-0.01, 0.01, 0.0], [0.0, 0.0, 0.03]])
    wk = np.array([[0.0, 0.002, 0.0], [0.001, 0.0, 0.0], [0.0, 0.0, -0.003]])
    Rk = np.array([3.0, 3.2, 2.5])
    f1, F, M, st = oracle.psm_step(shape, f, 0.6, (0, 0, 0), None, xk, vk, wk, Rk, trt=trt)   # Eq. 33 with BGK or TRT
    assert st == 0
    assert abs(f1.sum() - f.sum()) < 1e-12 * f.sum()
    assert np.abs(F).min() > 1e-5
    assert np.abs((momentum(f1) - momentum(f)) + F.sum(0)).max() < 1e-12


def test_force_identity_single_cell_sum():
    # G21: sum_i Omega^s c_i = rho (u_k - u) for both readings of Eq. 34, so
    # F_k = - sum_cells B_k rho (u_k - u); rebuilt here from moments with numpy.
    shape = (12, 12, 12)
    rho, u = W.random_flow(shape, 9, amp=0.01)
    f = oracle.lbm_equilibrium(shape, rho, u)
    f = oracle.lbm_run(shape, f, 0.8, 3)                                      # off equilibrium
    xk, vk, wk, R, tau = np.array([5.7, 6.2, 5.9]), np.array([0.01, -0.02, 0.015]), np.array([0.001, 0.002, -0.001]), 3.1, 0.7
    f1, F, M, st = oracle.psm_step(shape, f, tau, (1, 1, 1), None, xk[None], vk[None], wk[None], [R])
    rho_c, u_c = oracle.lbm_moments(shape, f)
    z, y, x = np.meshgrid(np.arange(12), np.arange(12), np.arange(12), indexing="ij")
    d = np.stack([x.ravel() - xk[0], y.ravel() - xk[1], z.ravel() - xk[2]], 0)
    dist = np.sqrt((d ** 2).sum(0))
    beta = np.clip(((R + oracle.psm_rc()) - dist) / (2 * oracle.psm_rc()), 0, 1)
    B = beta * (tau - 0.5) / ((1 - beta) + (tau - 0.5))
    uk = vk[:, None] + np.cross(wk, d.T).T
    dF = -B * rho_c * (uk - u_c)
    assert np.abs(F[0] - dF.sum(1)).max() < 1e-13
    assert np.abs(M[0] - np.cross(d.T, dF.T).sum(0)).max() < 1e-12


def test_comoving_sphere_and_fluid_feel_nothing():
    # (xvi): fluid at uniform U and a sphere translating at U: zero force, fluid unchanged
    shape = (12, 12, 12)
    n = 12 ** 3
    U = np.array([0.03, -0.02, 0.01])
    f = oracle.lbm_equilibrium(shape, np.ones(n), np.tile(U[:, None], (1, n)))
    f1, F, M, st = oracle.psm_step(shape, f, 0.6, (0, 0, 0), None, [[6.3, 5.8, 6.1]], [U], [[0, 0, 0]], [3.5])
    assert np.abs(F).max() < 1e-13 and np.abs(M).max() < 1e-12      # rounding of ~200 cells
    assert np.abs(f1 - f).max() < 1e-15


def test_fixed_point_inside_solid():
    # G21: with B = 1 and f = feq(rho, u_k) the solid operator vanishes: the interior stays at u_k
    shape = (14, 14, 14)
    n = 14 ** 3
    U = np.array([0.02, 0.0, 0.0])
    f = oracle.lbm_equilibrium(shape, np.ones(n), np.tile(U[:, None], (1, n)))
    f1, F, M, st = oracle.psm_step(shape, f, 0.6, (0, 0, 0), None, [[7.0, 7.0, 7.0]], [U], [[0, 0, 0]], [5.0])
    assert np.abs(f1 - f).max() < 1e-15


def test_torque_opposes_spin():
    # G22: a sphere spinning in fluid at rest is braked: M_sf . omega < 0 (wrong sign in Eq. 35 flips it);
    # after a few steps the fluid next to the surface co-rotates.
    shape = (20, 20, 20)
    f = oracle.lbm_equilibrium(shape)
    xk, wk = np.array([[9.5, 9.5, 9.5]]), np.array([[0.0, 0.0, 0.004]])
    for _ in range(5):
        f, F, M, st = oracle.psm_step(shape, f, 0.6, (0, 0, 0), None, xk, [[0, 0, 0]], wk, [5.0])
        assert M[0, 2] < 0 and abs(M[0, 0]) < 1e-12 and abs(M[0, 1]) < 1e-12
        assert np.abs(F).max() < 1e-12                      # symmetric set-up: no net force
    rho, u = oracle.lbm_moments(shape, f)
    ux = u[0].reshape(20, 20, 20)
    # node (x=9, y=14, z=9): r - r_k = (.., +4.5, ..) lies inside the solid -> u_x = (w x d)_x = -w_z d_y < 0
    assert ux[9, 14, 9] < -0.01 and ux[9, 5, 9] > 0.01


def _cell_terms(shape, f, tau, xk, vk, wk, R):
    """-B rho (u_k - u) per cell of one solid from the moments, in numpy (the identity of G21; pinned on its own by
    test_force_identity_single_cell_sum) -> dF [3, N], beta [N]"""
    nx, ny, nz = shape
    rho_c, u_c = oracle.lbm_moments(shape, f)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    d = np.stack([x.ravel() - xk[0], y.ravel() - xk[1], z.ravel() - xk[2]], 0)
    beta = np.clip(((R + oracle.psm_rc()) - np.sqrt((d ** 2).sum(0))) / (2 * oracle.psm_rc()), 0, 1)
    B = beta * (tau - 0.5) / ((1 - beta) + (tau - 0.5))
    uk = np.asarray(vk)[:, None] + np.cross(wk, d.T).T
    return -B * rho_c * (uk - u_c), beta


def test_two_lowest_ids_kept_and_flag_raised():
    # G24 (n_s = 2): a cell cut by three solids keeps the two LOWEST ids and raises status bit 2.
    # Solids 0 and 1 (R = 3) overlap around (8, 8, 8); solid 2 (R = 1.2) sits inside their intersection, so every
    # cell it cuts is already taken by 0 and 1: it is dropped everywhere.  The step must then equal, bit for bit,
    # the step without solid 2, and solid 2 feels nothing.  (Keeping the two highest ids instead gives F_2 != 0.)
    shape = (16, 16, 16)
    rho, u = W.random_flow(shape, 12, amp=0.01)
    f = oracle.lbm_equilibrium(shape, rho, u)
    xk = np.array([[7.0, 8.0, 8.0], [9.0, 8.0, 8.0], [8.0, 8.0, 8.0]])
    vk = np.array([[0.01, 0.0, 0.0], [-0.01, 0.005, 0.0], [0.0, 0.02, -0.01]])
    wk = np.array([[0.0, 0.0, 0.001], [0.002, 0.0, 0.0], [0.0, 0.003, 0.0]])
    Rk = np.array([3.0, 3.0, 1.2])
    f3, F3, M3, st3 = oracle.psm_step(shape, f, 0.6, (1, 1, 1), None, xk, vk, wk, Rk)
    f2, F2, M2, st2 = oracle.psm_step(shape, f, 0.6, (1, 1, 1), None, xk[:2], vk[:2], wk[:2], Rk[:2])
    assert st3 & 2 and st2 == 0
    assert np.array_equal(f3, f2)
    assert np.array_equal(F3[:2], F2) and np.array_equal(M3[:2], M2)
    assert np.all(F3[2] == 0.0) and np.all(M3[2] == 0.0)
    assert np.abs(F2).min() > 1e-6                              # the kept solids do exchange momentum
    # the same three solids renumbered so that the small one has the lowest id: now it is kept (with the lower of
    # the two large ones) and the highest id loses exactly the cells the small one cuts
    perm = [2, 0, 1]
    fp, Fp, Mp, stp = oracle.psm_step(shape, f, 0.6, (1, 1, 1), None, xk[perm], vk[perm], wk[perm], Rk[perm])
    assert stp & 2
    dF_small, beta_small = _cell_terms(shape, f, 0.6, xk[2], vk[2], wk[2], Rk[2])
    dF_big, beta_big = _cell_terms(shape, f, 0.6, xk[1], vk[1], wk[1], Rk[1])
    assert np.abs(Fp[0] - dF_small.sum(1)).max() < 1e-14                              # small one: all of its cells
    assert np.abs(Fp[1] - F2[0]).max() == 0.0                                         # the lower large one: untouched
    lost = beta_small > 0
    assert lost.sum() >= 7
    assert np.abs(Fp[2] - dF_big[:, ~lost].sum(1)).max() < 1e-14                      # the higher large one: minus those cells
    assert np.abs(dF_big[:, lost].sum(1)).max() > 1e-5                                # (and they matter)


def test_coupled_driver_buoyant_sphere_sinks_and_neutral_floats():
    # Eq. 56 / G27: density ratio 1 -> no net force at rest; ratio 1.5 -> accelerates along g with
    # a(0) = (1 - rho_f/rho_p) g and is then slowed by the fluid (|v| < free-fall value).
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(24, 24, 48), R=4.0, z0=30.0, g=1e-3)
    f0 = oracle.lbm_equilibrium(lbm["shape"])
    d = oracle.Dem(pd, x, v, w, R, pairs_mode="brute")
    assert abs(d.a[0, 2] + (1 - 1 / 1.5) * 1e-3) < 1e-18
    c = oracle.Coupled(lbm, cpl, d, f0)
    c.step(60)
    free = -(1 - 1 / 1.5) * 1e-3 * 60
    assert free < d.v[0, 2] < 0.3 * free * 0 - 1e-4 and d.x[0, 2] < 30.0
    assert c.F_sf[0, 2] > 0                                  # drag points up


# ---------------------------------------------------------------- subdivision solid fraction (Eq. 38)
def test_subdivision_fraction_limits_and_plane_cut():
    # far inside 1, far outside 0, values are multiples of 1/N; a (nearly) plane surface through the cell centre,
    # normal along an axis, leaves exactly half of the evenly spread points inside
    assert oracle.psm_beta_subdiv([0.3, -0.2, 0.1], 4.0) == 1.0
    assert oracle.psm_beta_subdiv([5.0, 0.0, 0.0], 4.0) == 0.0
    b = oracle.psm_beta_subdiv([3.7, 0.4, -0.3], 4.0)
    assert 0.0 < b < 1.0 and abs(b * 1000 - round(b * 1000)) < 1e-9
    R = 1.0e6
    for ax in range(3):
        d = [0.0, 0.0, 0.0]; d[ax] = R
        assert oracle.psm_beta_subdiv(d, R) == 0.5
        d[ax] = R - 0.2                                        # plane at +0.2 from the centre: layers at -0.45..0.15 inside
        assert abs(oracle.psm_beta_subdiv(d, R) - 0.7) < 1e-12
    # more points per direction: the same cut converges to the exact slab fraction 0.5 + 0.2
    assert abs(oracle.psm_beta_subdiv([R - 0.2, 0, 0], R, 40) - 0.7) <= 1.0 / 40


def test_subdivision_fraction_integrates_to_the_sphere_volume():
    # sum_j beta_j dx^3 is a midpoint-rule quadrature of the sphere volume on a 0.1 dx grid: within 0.2 %,
    # an order of magnitude closer than the distance-based estimate (3 %, G25)
    for R, xk in ((4.0, (10.3, 11.1, 9.7)), (6.0, (12.0, 12.5, 11.9)), (2.5, (11.27, 12.4, 12.9))):
        s = oracle.psm_beta_sum((24, 24, 24), (1, 1, 1), np.array(xk), R, subdiv=10)
        assert abs(s / (4 / 3 * np.pi * R ** 3) - 1.0) < 0.002


def test_subdivision_fraction_has_the_symmetry_of_the_lattice():
    # a sphere centred on a node: beta depends on |dx|, |dy|, |dz| only and is symmetric under their permutation
    for d in ([3.0, 2.0, 1.0], [3.6, 1.0, 0.0], [2.0, 2.0, 2.6]):
        ref = oracle.psm_beta_subdiv(d, 4.0)
        for perm in ((0, 1, 2), (1, 2, 0), (2, 0, 1), (0, 2, 1)):
            for sg in ((1, 1, 1), (-1, 1, -1), (1, -1, -1)):
                assert oracle.psm_beta_subdiv([sg[i] * d[perm[i]] for i in range(3)], 4.0) == ref


def test_subdivision_psm_step_budget_and_no_force_when_comoving():
    shape = (16, 14, 12)
    U = np.array([0.02, -0.01, 0.015])
    f = oracle.lbm_equilibrium(shape, None, np.tile(U[:, None], (1, 16 * 14 * 12)))
    xk = np.array([[5.2, 6.1, 5.7]]); Rk = np.array([3.0])
    f1, F, M, st = oracle.psm_step(shape, f, 0.6, (0, 0, 0), None, xk, U[None, :], np.zeros((1, 3)), Rk, subdiv=10)
    assert np.abs(F).max() < 1e-14 and np.abs(f1 - f).max() < 1e-15          # co-moving: nothing happens (to rounding)
    rho, u = W.random_flow(shape, 2, amp=0.01)
    f = oracle.lbm_equilibrium(shape, rho, u)
    f1, F, M, st = oracle.psm_step(shape, f, 0.6, (0, 0, 0), None, xk, np.array([[0.02, 0.0, -0.01]]), np.zeros((1, 3)), Rk,
                                   subdiv=10)
    assert np.abs((momentum(f1) - momentum(f)) + F.sum(0)).max() < 1e-12     # fluid momentum budget = -F
