"""CPU oracle for the LEDDS hot path (arxiv 2512.04997) -- TEST INFRASTRUCTURE.

Thin ctypes loader for oracle/liboracle.so (plain C, fp64, built by
oracle/build.py) plus the step drivers that put the C routines in the order
PAPER.md Table 1 gives.  Nothing here imports, calls or
shares code with the CUDA path (paper_2512_04997_b200/).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_up = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")


class DemParams(C.Structure):
    """Mirror of orc_dem_params (oracle/dem.c)."""
    _fields_ = [("n", C.c_int), ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("bc", C.c_int * 3),
                ("v_wall", C.c_double * 18), ("cell", C.c_double), ("dt", C.c_double), ("g", C.c_double * 3),
                ("density", C.c_double), ("kn", C.c_double), ("kt", C.c_double), ("restitution", C.c_double),
                ("mu", C.c_double), ("kn_w", C.c_double), ("kt_w", C.c_double), ("restitution_w", C.c_double),
                ("mu_w", C.c_double), ("model", C.c_int), ("young", C.c_double), ("poisson", C.c_double),
                ("young_w", C.c_double), ("poisson_w", C.c_double)]


def dem_params(d: dict) -> DemParams:
    """Build DemParams from the plain dict the workload generators return."""
    p = DemParams()
    p.n = int(d["n"])
    p.lo[:] = d["lo"]; p.hi[:] = d["hi"]; p.bc[:] = d["bc"]
    p.v_wall[:] = list(np.asarray(d.get("v_wall", np.zeros(18)), dtype=np.float64).ravel())
    p.cell = d["cell"]; p.dt = d["dt"]; p.g[:] = d["g"]; p.density = d["density"]
    p.kn = d["kn"]; p.kt = d["kt"]; p.restitution = d["restitution"]; p.mu = d["mu"]
    p.kn_w = d.get("kn_w", d["kn"]); p.kt_w = d.get("kt_w", d["kt"])
    p.restitution_w = d.get("restitution_w", d["restitution"]); p.mu_w = d.get("mu_w", d["mu"])
    p.model = int(d.get("model", 0))
    p.young = d.get("young", 0.0); p.poisson = d.get("poisson", 0.0)
    p.young_w = d.get("young_w", p.young); p.poisson_w = d.get("poisson_w", p.poisson)
    return p


def _sig(name, res, *args):
    fn = getattr(_lib, name)
    fn.restype = res
    fn.argtypes = list(args)
    return fn


_feq = _sig("orc_feq", C.c_double, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double)
_lattice = _sig("orc_lbm_lattice", None, _ip, _ip, _ip, _ip, _dp)
_lbm_eq = _sig("orc_lbm_equilibrium", None, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, _dp)
_lbm_mom = _sig("orc_lbm_moments", None, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp)
_lbm_run = _sig("orc_lbm_run", None, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _ip, _dp, _dp, _dp, C.c_int)
_trt_om = _sig("orc_trt_omega_minus", C.c_double, C.c_double)
_zeta = _sig("orc_dem_zeta", C.c_double, C.c_double)
_grid = _sig("orc_dem_grid", None, C.POINTER(DemParams), _ip, _dp)
_keys = _sig("orc_dem_keys", None, C.POINTER(DemParams), _dp, _up)
_order = _sig("orc_dem_order", None, C.c_int, _up, _up)
_pairs_brute = _sig("orc_dem_pairs_brute", C.c_int, C.POINTER(DemParams), _dp, _dp, _up, C.c_int)
_pairs_cells = _sig("orc_dem_pairs_cells", C.c_int, C.POINTER(DemParams), _dp, _dp, _up, _up, _up, C.c_int)
_forces = _sig("orc_dem_forces", None, C.POINTER(DemParams), _dp, _dp, _dp, _dp, C.c_int, _up, C.c_int, _up, _dp,
               C.c_double, _dp, _dp, _dp, _ip)
_advance = _sig("orc_dem_advance", None, C.POINTER(DemParams), _dp, _dp, _dp, _dp, _dp, _dp, _dp)
_kick = _sig("orc_dem_kick", None, C.POINTER(DemParams), _dp, _dp, _dp, C.c_void_p, C.c_void_p, _dp, _dp, _dp, _dp)
_psm_step = _sig("orc_psm_step", None, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, _ip, _dp, C.c_int, _dp, _dp, _dp, _dp,
                 _dp, _dp, _dp, _dp, _ip, _ip)
_psm_beta = _sig("orc_psm_beta", C.c_double, C.c_double, C.c_double)
_psm_B = _sig("orc_psm_B", C.c_double, C.c_double, C.c_double)
_psm_rc = _sig("orc_psm_rc", C.c_double)
_psm_beta_sum = _sig("orc_psm_beta_sum", C.c_double, C.c_int, C.c_int, C.c_int, _ip, _dp, C.c_double, C.c_int)
_psm_beta_subdiv = _sig("orc_psm_beta_subdiv", C.c_double, _dp, C.c_double, C.c_int)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# --------------------------------------------------------------------------- LBM
def lattice():
    cx, cy, cz, opp = (np.zeros(19, np.int32) for _ in range(4))
    t = np.zeros(19)
    _lattice(cx, cy, cz, opp, t)
    return cx, cy, cz, opp, t


def feq(i, rho, ux, uy, uz):
    return _feq(i, rho, ux, uy, uz)


def lbm_equilibrium(shape, rho=None, u=None):
    """shape = (nx, ny, nz); rho [N] or None; u [3, N] or None -> f [19, N]."""
    nx, ny, nz = shape
    f = np.empty((19, nx * ny * nz))
    rho = None if rho is None else _f64(rho).ravel()
    u = None if u is None else _f64(u).reshape(3, -1)
    _lbm_eq(nx, ny, nz, _ptr(rho), _ptr(u), f)
    return f


def lbm_moments(shape, f):
    nx, ny, nz = shape
    rho = np.empty(nx * ny * nz); u = np.empty((3, nx * ny * nz))
    _lbm_mom(nx, ny, nz, _f64(f), rho, u)
    return rho, u


def trt_omega_minus(omega_plus):
    """Eq. (31)"""
    return _trt_om(omega_plus)


def lbm_run(shape, f, tau, nsteps, bc=(0, 0, 0), u_wall=None, omega=None, omega_minus=None, trt=False):
    """nsteps collide-and-stream steps (Eq. 22-28); returns the new f [19, N].
    BGK unless trt (then omega_minus of Eq. 31) or an explicit omega_minus is given (TRT, Eq. 29-30)."""
    nx, ny, nz = shape
    f = _f64(f).copy()
    tmp = np.empty_like(f)
    uw = np.zeros(18) if u_wall is None else _f64(u_wall).ravel()
    om = (1.0 / tau) if omega is None else omega
    om_m = -1.0
    if omega_minus is not None:
        om_m = omega_minus
    elif trt:
        om_m = trt_omega_minus(om)
    _lbm_run(nx, ny, nz, om, om_m, np.asarray(bc, np.int32), uw, f, tmp, nsteps)
    return f


# --------------------------------------------------------------------------- DEM
def dem_zeta(eps):
    return _zeta(eps)


def dem_grid(pd):
    p = dem_params(pd)
    nc = np.zeros(3, np.int32); ih = np.zeros(3)
    _grid(C.byref(p), nc, ih)
    return nc, ih


class Dem:
    """DEM state advanced by the oracle, in the order of PAPER.md Table 1:
    integrate (18a) -> grid -> pair list -> forces -> reduce -> velocity update.

    History = last step's sorted pair list + delta_t per pair.
    pairs_mode: "cells" (uniform grid walk) or "brute" (O(N^2) definition).
    """

    def __init__(self, pd, x, v, w, radius, pairs_mode="cells", cap=None):
        self.pd = dict(pd)
        self.p = dem_params(pd)
        n = self.p.n
        self.n = n
        self.x = _f64(x).reshape(n, 3).copy(); self.v = _f64(v).reshape(n, 3).copy()
        self.w = _f64(w).reshape(n, 3).copy(); self.R = _f64(radius).reshape(n).copy()
        self.a = np.zeros((n, 3)); self.alpha = np.zeros((n, 3))
        self.vp = self.v.copy(); self.wp = self.w.copy()
        self.mode = pairs_mode
        self.cap = cap if cap is not None else 16 * n + 64
        self.pairs = np.zeros((0, 2), np.uint32); self.dt_hist = np.zeros((0, 3))
        self.status = np.zeros(1, np.int32)
        self.key = np.zeros(n, np.uint32); self.idx = np.zeros(n, np.uint32)
        self.F = np.zeros((n, 3)); self.M = np.zeros((n, 3))
        # a(0), alpha(0) from the contacts of the initial state; delta_t starts at 0
        self.contacts(0.0, self.v, self.w)
        v0, w0 = self.v.copy(), self.w.copy()      # throw-away: only a', alpha' of (18b), (19c) are kept
        _kick(C.byref(self.p), self.R, self.F, self.M, None, None, v0, w0, self.a, self.alpha)

    def contacts(self, dt_hist, v, w):
        """grid -> pair list -> forces; updates history; returns F, M."""
        p = self.p
        _keys(C.byref(p), self.x, self.key)
        _order(self.n, self.key, self.idx)
        buf = np.zeros((self.cap, 2), np.uint32)
        if self.mode == "brute":
            npairs = _pairs_brute(C.byref(p), self.x, self.R, buf, self.cap)
        else:
            npairs = _pairs_cells(C.byref(p), self.x, self.R, self.key, self.idx, buf, self.cap)
        if npairs > self.cap:
            raise RuntimeError("oracle pair capacity exceeded")
        pairs = np.ascontiguousarray(buf[:npairs])
        new_dt = np.zeros((max(npairs, 1), 3))
        prev_pairs = self.pairs if len(self.pairs) else np.zeros((1, 2), np.uint32)
        prev_dt = self.dt_hist if len(self.dt_hist) else np.zeros((1, 3))
        pp = pairs if npairs else np.zeros((1, 2), np.uint32)
        _forces(C.byref(p), self.x, _f64(v), _f64(w), self.R, npairs, pp, len(self.pairs), prev_pairs, prev_dt,
                dt_hist, new_dt, self.F, self.M, self.status)
        self.pairs = pairs
        self.dt_hist = np.ascontiguousarray(new_dt[:npairs])
        return self.F, self.M

    def advance(self):
        _advance(C.byref(self.p), self.x, self.v, self.w, self.a, self.alpha, self.vp, self.wp)

    def kick(self, f_ext=None, m_ext=None):
        fe = None if f_ext is None else _f64(f_ext)
        me = None if m_ext is None else _f64(m_ext)
        _kick(C.byref(self.p), self.R, self.F, self.M, _ptr(fe), _ptr(me), self.v, self.w, self.a, self.alpha)

    def step(self, nsteps=1, f_ext=None, m_ext=None):
        for _ in range(nsteps):
            self.advance()
            self.contacts(self.p.dt, self.vp, self.wp)
            self.kick(f_ext, m_ext)


# --------------------------------------------------------------------------- coupling
def psm_rc():
    return _psm_rc()


def psm_beta(Rk, dist):
    return _psm_beta(Rk, dist)


def psm_B(beta, tau):
    return _psm_B(beta, tau)


def psm_beta_sum(shape, bc, xk, Rk, subdiv=0):
    return _psm_beta_sum(shape[0], shape[1], shape[2], np.asarray(bc, np.int32), _f64(xk), Rk, int(subdiv))


def psm_beta_subdiv(d, Rk, ns=10):
    """Eq. (38): d = r_j - r_k (cell centre minus sphere centre), ns points per direction."""
    return _psm_beta_subdiv(_f64(d), Rk, int(ns))


def psm_step(shape, f, tau, bc, u_wall, xk, vk, wk, Rk, trt=False, subdiv=0):
    """One PSM collide-and-stream step in lattice units (Eq. 32-42).
    Returns f_new [19,N], F [np,3], M [np,3], status."""
    nx, ny, nz = shape
    n = len(Rk)
    f = _f64(f)
    f_out = np.empty_like(f)
    F = np.zeros((max(n, 1), 3)); M = np.zeros((max(n, 1), 3))
    slots = np.empty(2 * nx * ny * nz, np.int32)
    status = np.zeros(1, np.int32)
    uw = np.zeros(18) if u_wall is None else _f64(u_wall).ravel()
    pad = lambda a, k: _f64(a).reshape(-1) if n else np.zeros(k)
    _psm_step(nx, ny, nz, tau, trt_omega_minus(1.0 / tau) if trt else -1.0, int(subdiv), np.asarray(bc, np.int32), uw, n, pad(xk, 3), pad(vk, 3), pad(wk, 3), pad(Rk, 1),
              f, f_out, F, M, slots, status)
    return f_out, F[:n], M[:n], int(status[0])


class Coupled:
    """Coupled LBM-DEM step (SURVEY (c.3)).

    lbm: dict(shape, tau, bc, u_wall); cpl: dict(n_sub, dx, rho_f, origin).
    Lattice node i sits at origin + i*dx in DEM length units; the LBM time step
    is n_sub * dt.  F_sf, M_sf of the previous LBM step are held during the
    sub-steps; the last sub-step's corrector uses the new ones.
    Pins (tests/test_oracle_coupled.py): the step does not depend on the units it is
    posed in (dx, Dt, rho_f, origin: every conversion exponent), and the velocity after
    two steps with n_sub = 4 is the closed form of "F_sf held, refreshed in the last kick".
    """

    def __init__(self, lbm, cpl, dem: Dem, f):
        self.lbm, self.cpl, self.dem = lbm, cpl, dem
        self.f = _f64(f).copy()
        self.F_sf = np.zeros((dem.n, 3)); self.M_sf = np.zeros((dem.n, 3))
        self.status = 0

    def step(self, nsteps=1):
        d, cpl, lbm = self.dem, self.cpl, self.lbm
        dx, rho_f, n_sub = cpl["dx"], cpl["rho_f"], cpl["n_sub"]
        org = np.asarray(cpl.get("origin", (0.0, 0.0, 0.0)))
        Dt = n_sub * d.p.dt
        for _ in range(nsteps):
            for s in range(n_sub):
                d.advance()
                d.contacts(d.p.dt, d.vp, d.wp)
                if s < n_sub - 1:
                    d.kick(self.F_sf, self.M_sf)
            xk = (d.x - org[None, :]) / dx
            vk = d.vp * (Dt / dx)
            wk = d.wp * Dt
            Rk = d.R / dx
            self.f, F, M, st = psm_step(lbm["shape"], self.f, lbm["tau"], lbm["bc"], lbm.get("u_wall"), xk, vk, wk, Rk,
                                        trt=bool(lbm.get("collision", 0)), subdiv=10 if cpl.get("solid_fraction", 0) else 0)
            self.status |= st
            self.F_sf = F * (rho_f * dx ** 4 / Dt ** 2)
            self.M_sf = M * (rho_f * dx ** 5 / Dt ** 2)
            d.kick(self.F_sf, self.M_sf)
