"""Pins for the unit conversions of oracle.Coupled (reading G32, Eq. 41-42) and for holding
F_sf during sub-steps (G28).  CPU only.

The same physical problem is posed twice: once in lattice units (dx = rho_f = Dt = 1, origin 0) and once in other
units of length L, time T and mass Mu = rho_f L^3, with the lattice node (0,0,0) somewhere else in the DEM frame.
Every DEM quantity of the second problem is the first one's times its dimension's factor; the lattice does not know
about units.  The two runs must then agree after converting back: a wrong exponent in rho_f dx^4 / Dt^2 (force),
rho_f dx^5 / Dt^2 (torque), Dt / dx (velocity), Dt (spin) or a dropped origin shows up at first order."""
import numpy as np
import pytest

import oracle
import workloads as W


def posed_in_units(L, T, rho_f, origin, n_sub, steps, two=False):
    lbm, cpl, pd, x, v, w, R = W.cfg3_settling(shape=(24, 20, 40), R=3.6, z0=22.0, g=2e-3)
    if two:                                                   # a second sphere touching the first: contact forces too
        x = np.array([[11.0, 10.0, 22.0], [15.3, 11.0, 26.3]]); R = np.array([3.6, 2.9])
        pd = dict(pd, n=2)
    n = len(R)
    v = np.tile(np.array([[0.004, -0.002, 0.0]]), (n, 1)); w = np.tile(np.array([[0.001, 0.002, -0.0015]]), (n, 1))
    Mu = rho_f * L ** 3
    org = np.asarray(origin, float)
    pdB = dict(pd)
    pdB.update(lo=tuple(org + L * np.asarray(pd["lo"])), hi=tuple(org + L * np.asarray(pd["hi"])), cell=pd["cell"] * L,
               dt=T / n_sub, g=tuple(np.asarray(pd["g"]) * L / T ** 2), density=pd["density"] * Mu / L ** 3)
    for k in ("kn", "kt", "kn_w", "kt_w"):
        pdB[k] = pd[k] * Mu / T ** 2
    cplB = dict(n_sub=n_sub, dx=L, rho_f=rho_f, origin=tuple(org))
    d = oracle.Dem(pdB, org + L * x, v * L / T, w / T, R * L, pairs_mode="brute")
    Fc0 = d.F * T ** 2 / (Mu * L)                              # contact forces of the initial state
    c = oracle.Coupled(lbm, cplB, d, oracle.lbm_equilibrium(lbm["shape"]))
    c.step(steps)
    # back to lattice units
    return dict(x=(d.x - org) / L, v=d.v * T / L, w=d.w * T, F=c.F_sf * T ** 2 / (Mu * L), M=c.M_sf * T ** 2 / (Mu * L ** 2),
                f=c.f, Fc=Fc0)


@pytest.mark.parametrize("n_sub", [1, 4])
@pytest.mark.parametrize("two", [False, True])
def test_coupled_step_does_not_depend_on_the_units_it_is_posed_in(n_sub, two):
    steps = 12
    a = posed_in_units(1.0, 1.0, 1.0, (0.0, 0.0, 0.0), n_sub, steps, two)
    assert np.abs(a["F"]).max() > 1e-4 and np.abs(a["M"]).max() > 1e-6 and np.abs(a["v"]).max() > 1e-3
    if two:
        assert np.abs(a["Fc"]).max() > 1e-6                    # the spheres do touch (and part within the run)
    # powers of two (every scaling exact, only the shift by the origin rounds) and a generic SI-like set
    for L, T, rho_f, org, tol in ((0.5, 0.25, 2.0, (3.0, -1.5, 0.25), 1e-12), (3.0e-4, 7.0e-4, 998.2, (0.0123, -0.4, 1.7), 1e-9)):
        b = posed_in_units(L, T, rho_f, org, n_sub, steps, two)
        for k in ("x", "v", "w", "F", "M", "f"):
            scale = np.abs(a[k]).max()
            assert np.abs(b[k] - a[k]).max() <= tol * scale, (k, L, np.abs(b[k] - a[k]).max() / scale)


def test_hydrodynamic_force_is_held_during_the_sub_steps():
    # G28: with n_sub sub-steps the DEM sees the F_sf of the previous LBM step in every kick but
    # the last, which takes the new one.  A force-free neutrally buoyant sphere pushed by a uniform stream: after
    # ONE coupled step its velocity is dt_p/2 (a0 + a_last) summed over the sub-steps, with F_sf(previous) = 0 in
    # all kicks but the last: v = (Dt / n_sub) / 2 * F_sf / m, not Dt/2 * F_sf / m.
    shape = (20, 20, 20)
    n = 20 ** 3
    U = np.array([0.02, 0.0, 0.0])
    f0 = oracle.lbm_equilibrium(shape, np.ones(n), np.tile(U[:, None], (1, n)))
    R, n_sub = 3.5, 4
    pd = W.dem_defaults(1, (-0.5,) * 3, (19.5,) * 3, (0, 0, 0), cell=2 * R + 1, dt=1.0 / n_sub, g=(0, 0, 0), density=1.0, kn=1.0,
                        restitution=1.0, mu=0.0)
    d = oracle.Dem(pd, [[9.6, 10.2, 9.9]], [[0, 0, 0]], [[0, 0, 0]], [R], pairs_mode="brute")
    c = oracle.Coupled(dict(shape=shape, tau=0.7, bc=(0, 0, 0), u_wall=None), dict(n_sub=n_sub, dx=1.0, rho_f=1.0), d, f0)
    c.step(1)
    m = 4.0 / 3.0 * np.pi * R ** 3
    F1 = c.F_sf[0].copy()
    assert F1[0] > 1e-3
    v1 = d.v[0].copy()
    assert np.abs(v1 - 0.5 * (1.0 / n_sub) * F1 / m).max() < 1e-15
    assert np.abs(d.x[0] - [9.6, 10.2, 9.9]).max() == 0.0       # it has not moved yet: v was 0 in every drift
    # second step: the first n_sub - 1 kicks see F1 on both sides of Eq. (18c) (held), the last one F1 and the new F2
    c.step(1)
    F2 = c.F_sf[0]
    dtp = 1.0 / n_sub
    assert np.abs(F2 - F1).max() > 1e-6
    assert np.abs(d.v[0] - (v1 + (n_sub - 1) * dtp * F1 / m + 0.5 * dtp * (F1 + F2) / m)).max() < 1e-15
