"""Pins for oracle/lbm.c against what the paper and the mathematics fix
(SURVEY 8(c.5) ii, iii, vi, vii, viii; readings G17-G19, G29).  CPU only."""
import numpy as np
import pytest

import oracle
import workloads as W


def test_lattice_isotropy_and_opposites():
    # G18: sum t = 1, sum t c = 0, sum t c c = I/3 (c_s^2 = 1/3), opp reverses c
    cx, cy, cz, opp, t = oracle.lattice()
    c = np.stack([cx, cy, cz], 1).astype(float)
    assert abs(t.sum() - 1.0) < 1e-15
    assert np.abs((t[:, None] * c).sum(0)).max() < 1e-16
    assert np.allclose(np.einsum("i,ia,ib->ab", t, c, c), np.eye(3) / 3.0, atol=1e-15)
    # fourth-order isotropy: sum t c_a c_b c_c c_d = (1/9)(d_ab d_cd + d_ac d_bd + d_ad d_bc)
    T4 = np.einsum("i,ia,ib,ic,id->abcd", t, c, c, c, c)
    I = np.eye(3)
    ref = (np.einsum("ab,cd->abcd", I, I) + np.einsum("ac,bd->abcd", I, I) + np.einsum("ad,bc->abcd", I, I)) / 9.0
    assert np.allclose(T4, ref, atol=1e-15)
    assert np.all(c[opp] == -c)
    assert len({tuple(v) for v in c.astype(int)}) == 19 and np.all(np.abs(c).sum(1) <= 2)


def test_equilibrium_moments():
    # Eq. (22) applied to Eq. (28) returns rho and rho*u exactly; second moment = rho(c_s^2 I + u u)
    cx, cy, cz, opp, t = oracle.lattice()
    rho, u = 1.07, np.array([0.03, -0.02, 0.05])
    fe = np.array([oracle.feq(i, rho, *u) for i in range(19)])
    c = np.stack([cx, cy, cz], 1).astype(float)
    assert abs(fe.sum() - rho) < 1e-15
    assert np.abs(fe @ c - rho * u).max() < 1e-16
    P = np.einsum("i,ia,ib->ab", fe, c, c)
    assert np.allclose(P, rho * (np.eye(3) / 3 + np.outer(u, u)), atol=1e-15)


def test_uniform_equilibrium_is_fixed_point():
    shape = (6, 5, 4)
    n = 120
    u = np.tile(np.array([[0.03], [-0.01], [0.02]]), (1, n))
    f0 = oracle.lbm_equilibrium(shape, np.full(n, 1.1), u)
    f1 = oracle.lbm_run(shape, f0, 0.7, 7)
    assert np.abs(f1 - f0).max() < 1e-15


@pytest.mark.parametrize("bc,steps", [((0, 0, 0), 6), ((1, 1, 1), 120), ((0, 1, 0), 120)])
def test_pure_streaming_is_a_permutation(bc, steps):
    # omega = 0: populations are only moved, so the multiset of values never changes; in a periodic
    # cube the field returns bit for bit after n steps; with walls every population retraces its
    # path between two bounces (length L <= n, period 2L), so after 2*lcm(1..6) = 120 steps.
    n = 6
    shape = (n, n, n)
    f0 = np.random.default_rng(0).random((19, n ** 3))
    f1 = oracle.lbm_run(shape, f0, 1.0, 1, bc=bc, omega=0.0)
    assert np.array_equal(np.sort(f1.ravel()), np.sort(f0.ravel()))
    assert not np.array_equal(f1, f0)
    fn = oracle.lbm_run(shape, f0, 1.0, steps, bc=bc, omega=0.0)
    assert np.array_equal(fn, f0)


def test_streaming_moves_to_the_neighbour_it_travels_to():
    # Eq. (25): a marker in direction i at r appears at r + c_i
    cx, cy, cz, opp, t = oracle.lattice()
    shape = (5, 6, 7)
    nx, ny, nz = shape
    for i in range(19):
        f0 = np.ones((19, nx * ny * nz))
        f0[i, (3 * ny + 2) * nx + 1] = 2.0
        f1 = oracle.lbm_run(shape, f0, 1.0, 1, omega=0.0)
        q, c = np.nonzero(f1 == 2.0)
        assert len(q) == 1 and q[0] == i
        assert c[0] == ((3 + cz[i]) * ny + (2 + cy[i])) * nx + (1 + cx[i])


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1), (1, 0, 1)])
def test_mass_conservation(bc):
    shape = (12, 10, 8)
    rho, u = W.random_flow(shape, 3)
    f = oracle.lbm_equilibrium(shape, rho, u)
    m0 = f.sum()
    f = oracle.lbm_run(shape, f, 0.6, 100, bc=bc)
    assert abs(f.sum() - m0) / m0 <= 1e-13


def test_momentum_conservation_periodic():
    shape = (8, 8, 8)
    cx, cy, cz, opp, t = oracle.lattice()
    rho, u = W.random_flow(shape, 5)
    f = oracle.lbm_equilibrium(shape, rho, u)
    c = np.stack([cx, cy, cz], 1).astype(float)
    p0 = f.sum(1) @ c
    f = oracle.lbm_run(shape, f, 0.8, 50)
    assert np.abs(f.sum(1) @ c - p0).max() < 1e-12


@pytest.mark.parametrize("plane", ["xy", "yz", "zx"])
def test_taylor_green_decay(plane):
    # G29: E(t)/E(0) = exp(-4 nu k^2 t), nu = (tau - 1/2)/3 (Eq. 27).  The equilibrium start
    # lacks the viscous stress, which costs ~1 % of E in the first steps; after
    # that the decay RATE must be the closed form's (0.5 %), and E itself stays within 2 %.
    n, tau = 32, 0.6
    shape = (n, n, n)
    rho, u = W.tgv(shape, 0.02, 1.0, plane)
    f = oracle.lbm_equilibrium(shape, rho, u)
    e0 = (u ** 2).sum()
    f = oracle.lbm_run(shape, f, tau, 100)
    e1 = (oracle.lbm_moments(shape, f)[1] ** 2).sum()
    f = oracle.lbm_run(shape, f, tau, 200)
    e2 = (oracle.lbm_moments(shape, f)[1] ** 2).sum()
    k = 2 * np.pi / n
    rate = 4.0 * (tau - 0.5) / 3.0 * k * k
    assert abs(np.log(e1 / e2) / 200.0 / rate - 1.0) < 0.005
    assert abs(e2 / e0 / np.exp(-rate * 300) - 1.0) < 0.02


def test_taylor_green_closed_form_value_for_config2():
    # the number config 2 is checked against: exp(-4 nu k^2 t) at 128^3, tau 0.6, t = 1000 (golden file)
    import os
    val = float(open(os.path.join(os.path.dirname(__file__), "golden", "tgv_config2.txt")).read().split()[0])
    assert abs(val - np.exp(-4.0 * (0.1 / 3.0) * (2 * np.pi / 128) ** 2 * 1000)) < 5e-6


def test_couette_profile():
    # G19: halfway bounce-back, walls half a spacing outside the outermost nodes; steady state is
    # the linear profile u_x(z) = U_lo + (U_hi - U_lo)(z + 1/2)/nz, exact for BGK up to rounding.
    shape = (2, 2, 9)
    nz = 9
    uw = np.zeros((3, 2, 3)); uw[2, 0, 0] = -0.03; uw[2, 1, 0] = 0.05
    f = oracle.lbm_equilibrium(shape)
    f = oracle.lbm_run(shape, f, 1.0, 3000, bc=(0, 0, 1), u_wall=uw)
    rho, u = oracle.lbm_moments(shape, f)
    ux = u[0].reshape(nz, 2, 2)[:, 0, 0]
    ref = -0.03 + 0.08 * (np.arange(nz) + 0.5) / nz
    assert np.abs(ux - ref).max() < 1e-10
    assert np.abs(u[1]).max() < 1e-14 and np.abs(u[2]).max() < 1e-12
    assert abs(f.sum() - 36.0) < 1e-10            # moving walls parallel to themselves add no mass


# ---------------------------------------------------------------- TRT (Eq. 29-31)
def test_trt_magic_parameter_is_three_sixteenths():
    # Eq. (31) is the statement (tau+ - 1/2)(tau- - 1/2) = 3/16 for every tau+ (the value of [57])
    for tau in (0.51, 0.55, 0.6, 0.8, 1.0, 1.7):
        om = oracle.trt_omega_minus(1.0 / tau)
        assert abs((tau - 0.5) * (1.0 / om - 0.5) - 3.0 / 16.0) < 1e-15


def test_trt_with_equal_rates_is_bgk():
    # Eq. (30) with tau- = tau+: f+ + f- = f, so the model is Eq. (26)
    shape = (9, 8, 7)
    rho, u = W.random_flow(shape, 5)
    f = oracle.lbm_equilibrium(shape, rho, u) * (1.0 + 0.01 * np.random.default_rng(3).standard_normal((19, 9 * 8 * 7)))
    uw = np.zeros((3, 2, 3)); uw[2, 1, 0] = 0.04
    for bc in ((0, 0, 0), (0, 0, 1)):
        a = oracle.lbm_run(shape, f, 0.7, 5, bc=bc, u_wall=uw)
        b = oracle.lbm_run(shape, f, 0.7, 5, bc=bc, u_wall=uw, omega_minus=1.0 / 0.7)
        assert np.abs(a - b).max() < 1e-15


def test_trt_conserves_mass_and_momentum_and_keeps_equilibrium():
    shape = (8, 6, 10)
    rho, u = W.random_flow(shape, 6)
    f = oracle.lbm_equilibrium(shape, rho, u)
    g = oracle.lbm_run(shape, f, 0.58, 20, trt=True)
    cx, cy, cz, opp, t = oracle.lattice()
    assert abs(g.sum() - f.sum()) < 1e-12 * f.sum()
    for c in (cx, cy, cz):
        assert abs((g.sum(1) * c).sum() - (f.sum(1) * c).sum()) < 1e-12
    fe = oracle.lbm_equilibrium(shape, np.full(8 * 6 * 10, 1.1), np.tile(np.array([[0.02], [-0.01], [0.015]]), (1, 480)))
    assert np.abs(oracle.lbm_run(shape, fe, 0.58, 3, trt=True) - fe).max() < 1e-15


@pytest.mark.parametrize("tau", [0.6, 0.9])
def test_trt_viscosity_is_set_by_tau_plus_alone(tau):
    # Taylor-Green decay rate 2 nu k^2 (velocity) with nu = (tau+ - 1/2)/3, whatever tau-
    n = 32
    shape = (n, n, 4)
    rho, u = W.tgv(shape, 0.01, 1.0, "xy")
    f0 = oracle.lbm_equilibrium(shape, rho, u)
    k = 2 * np.pi / n
    for kw in (dict(trt=True), dict(omega_minus=1.3)):
        f = oracle.lbm_run(shape, f0, tau, 200, **kw)
        r1, u1 = oracle.lbm_moments(shape, f)
        rate = -np.log((u1 ** 2).sum() / (u ** 2).sum()) / 200
        assert abs(rate / (4 * (tau - 0.5) / 3 * k * k) - 1.0) < 0.02      # 1.2 % is the n = 32 discretisation error (BGK has it too)


def test_trt_odd_part_relaxes_with_tau_minus():
    # a population pair perturbed antisymmetrically (pure f-) at rest decays by the factor (1 - dt/tau-) per
    # collision; a symmetric perturbation (pure f+) by (1 - dt/tau+): distinguishes the two rates and their roles
    shape = (1, 1, 1)
    f0 = oracle.lbm_equilibrium(shape)
    om_p, om_m = 1.0 / 0.8, 0.37
    eps = 1e-3
    fa = f0.copy(); fa[1] += eps; fa[2] -= eps            # odd in (+x, -x): changes the momentum, so compare after removing
    g = oracle.lbm_run(shape, fa, 0.8, 1, omega_minus=om_m)   # the equilibrium shift: use the symmetric test for the even part
    fs = f0.copy(); fs[3] += eps; fs[4] += eps; fs[0] -= 2 * eps   # even in (+y, -y), mass kept, no momentum
    h = oracle.lbm_run(shape, fs, 0.8, 1, omega_minus=om_m)
    # periodic 1-cell box: streaming maps every population onto itself, so one step = one collision
    cx, cy, cz, opp, t = oracle.lattice()
    rho, ux = fa.sum(), (fa[:, 0] * cx).sum() / fa.sum()
    feq = np.array([oracle.feq(i, rho, ux, 0.0, 0.0) for i in range(19)])
    fm = 0.5 * (fa[1, 0] - fa[2, 0]); em = 0.5 * (feq[1] - feq[2])
    assert abs(0.5 * (g[1, 0] - g[2, 0]) - (fm - om_m * (fm - em))) < 1e-16
    feqs = np.array([oracle.feq(i, fs.sum(), 0.0, 0.0, 0.0) for i in range(19)])
    fp = 0.5 * (fs[3, 0] + fs[4, 0])
    assert abs(0.5 * (h[3, 0] + h[4, 0]) - (fp - om_p * (fp - feqs[3]))) < 1e-16


# ---------------------------------------------------------------- walls moving on two axes (reading G19)
def test_duct_with_all_four_walls_moving_along_its_axis_is_uniform_flow():
    # walls on y and z, all moving along the periodic x axis at the same U: f^eq(rho, U) is an exact fixed point
    # of velocity-modified halfway bounce-back (f_ibar^eq - f_i^eq = -6 t_i rho c_i.U), and a fluid started at
    # rest is dragged to u = (U, 0, 0) everywhere.  Links (+-1, +-1, 0) and (+-1, 0, +-1) cross one wall each.
    shape = (2, 6, 5)
    U = 0.04
    uw = np.zeros((3, 2, 3)); uw[1, :, 0] = U; uw[2, :, 0] = U
    n = 2 * 6 * 5
    fe = oracle.lbm_equilibrium(shape, np.ones(n), np.tile(np.array([[U], [0.0], [0.0]]), (1, n)))
    assert np.abs(oracle.lbm_run(shape, fe, 0.8, 5, bc=(0, 1, 1), u_wall=uw) - fe).max() < 1e-16
    f = oracle.lbm_run(shape, oracle.lbm_equilibrium(shape), 1.0, 2500, bc=(0, 1, 1), u_wall=uw)
    rho, u = oracle.lbm_moments(shape, f)
    assert np.abs(u[0] - U).max() < 1e-10 and np.abs(u[1]).max() < 1e-12 and np.abs(u[2]).max() < 1e-12
    assert abs(f.sum() - n) < 1e-10


def test_corner_link_crossing_two_moving_walls_takes_both_terms():
    # G19: "on a link crossing two walls use the sum of c_i.u_w over the crossed walls".  y walls slide along z,
    # z walls slide along y (and both along x).  At a corner node the links (0, +1, +1), (0, +1, -1), (0, -1, +1)
    # leave through the y-high wall, the y-high wall and the z-high wall: their terms 6 t rho (W + V), 6 t rho (-W)
    # and 6 t rho (-V) cancel only if the corner link carries BOTH walls' terms.  So total mass is conserved to
    # rounding with the sum reading, and drifts by O(t rho V) per corner node and step with any other reading
    # (one wall only, or the mean of the two).
    shape = (4, 6, 5)
    uw = np.zeros((3, 2, 3))
    uw[1, 0] = (0.01, 0.0, 0.03); uw[1, 1] = (-0.02, 0.0, -0.04)        # y walls: tangential = x, z
    uw[2, 0] = (0.02, -0.05, 0.0); uw[2, 1] = (0.0, 0.035, 0.0)         # z walls: tangential = x, y
    rho, u = W.random_flow(shape, 8, amp=0.01)
    f0 = oracle.lbm_equilibrium(shape, rho, u)
    m0 = f0.sum()
    f = f0
    for _ in range(6):
        f = oracle.lbm_run(shape, f, 0.7, 10, bc=(0, 1, 1), u_wall=uw)
        assert abs(f.sum() - m0) < 1e-13 * m0
    # one wall's term alone would lose 6 t rho V ~ 6/36 * 0.035 per corner node and step: 4 orders above the bound
    # and the fluid next to the y-high wall follows it in -z, next to the z-high wall in +y (signs of the terms)
    f = oracle.lbm_run(shape, oracle.lbm_equilibrium(shape), 0.7, 200, bc=(0, 1, 1), u_wall=uw)
    rho, u = oracle.lbm_moments(shape, f)
    uy, uz = u[1].reshape(5, 6, 4), u[2].reshape(5, 6, 4)
    assert uz[2, 5, 0] < -0.01 and uz[2, 0, 0] > 0.005 and uy[4, 3, 0] > 0.01 and uy[0, 3, 0] < -0.015
