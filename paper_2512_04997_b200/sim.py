"""Buffer-owning wrappers around the C ABI: allocate the device buffers the library asks for
(torch tensors), copy inputs in, call ledds_* and copy results out.  No arithmetic of the method
lives here; every step runs in the CUDA kernels behind include/ledds.h."""
import numpy as np
import torch

import paper_2512_04997_b200 as L


def _dev(a, dtype=torch.float64):
    """host array -> contiguous CUDA tensor (through pinned memory)"""
    t = torch.from_numpy(np.ascontiguousarray(a))
    if t.dtype != dtype:
        t = t.to(dtype)
    return t.pin_memory().to("cuda", non_blocking=True)


class Lbm:
    """D3Q19 lattice on the GPU (ledds_lbm_*; precision="f32" -> the ledds_lbm_*_f32 calls on float buffers)."""

    def __init__(self, lbm: dict, rho=None, u=None, f_canonical=None, precision="f64"):
        self.p = L.lbm_params(lbm)
        self.shape = tuple(lbm["shape"])
        self.N = self.shape[0] * self.shape[1] * self.shape[2]
        f32 = self.f32 = precision == "f32"
        if precision not in ("f64", "f32"):
            raise ValueError(precision)
        self.dtype = torch.float32 if f32 else torch.float64
        self._bytes, self._init, self._import, self._step, self._export = (
            (L.ledds_lbm_workspace_bytes_f32, L.ledds_lbm_init_f32, L.ledds_lbm_import_f32, L.ledds_lbm_step_f32,
             L.ledds_lbm_export_f32) if f32 else
            (L.ledds_lbm_workspace_bytes, L.ledds_lbm_init, L.ledds_lbm_import, L.ledds_lbm_step, L.ledds_lbm_export))
        self.f = torch.empty(self._bytes(self.p) // (4 if f32 else 8), dtype=self.dtype, device="cuda")
        rho_d = None if rho is None else _dev(rho, self.dtype).reshape(-1)
        u_d = None if u is None else _dev(u, self.dtype).reshape(-1)
        self.h = self._init(self.p, self.f, rho_d, u_d)
        if f_canonical is not None:
            self._import(self.h, self.f, _dev(f_canonical, self.dtype).reshape(-1))
        torch.cuda.current_stream().synchronize()     # rho_d / u_d may be freed after this

    def step(self, nsteps=1):
        self._step(self.h, self.f, nsteps)

    def export(self, want_f=True, want_moments=False):
        fc = torch.empty(19 * self.N, dtype=self.dtype, device="cuda") if want_f else None
        rho = torch.empty(self.N, dtype=self.dtype, device="cuda") if want_moments else None
        u = torch.empty(3 * self.N, dtype=self.dtype, device="cuda") if want_moments else None
        self._export(self.h, self.f, fc, rho, u)
        out = []
        if want_f:
            out.append(fc.cpu().numpy().reshape(19, self.N))
        if want_moments:
            out += [rho.cpu().numpy(), u.cpu().numpy().reshape(3, self.N)]
        return out[0] if len(out) == 1 else tuple(out)

    def __del__(self):
        try:
            L.ledds_lbm_destroy(self.h)
        except Exception:
            pass


class Dem:
    """Sphere DEM on the GPU (ledds_dem_*; precision="f32" -> the ledds_dem_*_f32 calls on float arrays).
    State tensors are [n,3] in particle order."""

    DEFAULTS = {}   # ledds_dem_params switches (no_single_block, cell_order, ...) for parameter dicts that do not name them: tests run every path

    def __init__(self, pd: dict, x, v, w, radius, precision="f64"):
        if precision not in ("f64", "f32"):
            raise ValueError(precision)
        self.pd = dict(pd)
        for key, val in Dem.DEFAULTS.items():
            self.pd.setdefault(key, val)
        self.p = L.dem_params(self.pd)
        self.f32 = precision == "f32"
        dt = self.dtype = torch.float32 if self.f32 else torch.float64
        self._bytes, self._init, self._step, self._query = (
            (L.ledds_dem_workspace_bytes_f32, L.ledds_dem_init_f32, L.ledds_dem_step_f32, L.ledds_dem_query_f32) if self.f32 else
            (L.ledds_dem_workspace_bytes, L.ledds_dem_init, L.ledds_dem_step, L.ledds_dem_query))
        n = self.n = self.p.n
        self.x, self.v, self.w = _dev(x, dt).reshape(n, 3), _dev(v, dt).reshape(n, 3), _dev(w, dt).reshape(n, 3)
        self.radius = _dev(radius, dt).reshape(n)
        self.a = torch.zeros(n, 3, dtype=dt, device="cuda")
        self.alpha = torch.zeros(n, 3, dtype=dt, device="cuda")
        sb, hb = self._bytes(self.p)
        self.scratch = torch.empty(sb, dtype=torch.uint8, device="cuda")
        self.history = torch.empty(hb, dtype=torch.uint8, device="cuda")
        self.status = torch.zeros(4, dtype=torch.int32, device="cuda")
        self.h = self._init(self.p, self.x, self.v, self.w, self.radius, self.a, self.alpha, self.history,
                            self.scratch, self.status)

    def step(self, nsteps=1, f_ext=None, m_ext=None):
        self._step(self.h, self.x, self.v, self.w, self.a, self.alpha, self.radius, f_ext, m_ext, self.history,
                   self.scratch, self.status, nsteps)

    def query(self, pair_cap=None):
        n = self.n
        cap = pair_cap if pair_cap is not None else 16 * n + 64
        idx = torch.empty(n, dtype=torch.int32, device="cuda"); key = torch.empty(n, dtype=torch.int32, device="cuda")
        pairs = torch.zeros(cap, 2, dtype=torch.int32, device="cuda")
        pdt = torch.zeros(cap, 3, dtype=self.dtype, device="cuda")
        npairs = torch.zeros(4, dtype=torch.int32, device="cuda")
        F = torch.empty(n, 3, dtype=self.dtype, device="cuda"); M = torch.empty(n, 3, dtype=self.dtype, device="cuda")
        self._query(self.h, self.history, self.scratch, idx, key, pairs, pdt, cap, npairs, F, M)
        k = int(npairs[0].item())
        if k > cap:
            raise L.LeddsError("pair_cap too small")
        u32 = lambda t: t.cpu().numpy().view(np.uint32)
        return dict(idx=u32(idx), key=u32(key), pairs=u32(pairs[:k]), pair_dt=pdt[:k].cpu().numpy(),
                    F=F.cpu().numpy(), M=M.cpu().numpy(), status=int(self.status[0].item()))

    def state(self):
        return {k: getattr(self, k).cpu().numpy() for k in ("x", "v", "w", "a", "alpha")}

    def __del__(self):
        try:
            L.ledds_dem_destroy(self.h)
        except Exception:
            pass


class Coupled:
    """Coupled LBM-DEM step on the GPU (ledds_coupled_step; ledds_coupled_step_f32 when the lattice is fp32)."""

    def __init__(self, lbm: Lbm, dem: Dem, cpl: dict, r_max: float):
        self.lbm, self.dem = lbm, dem
        self.c = L.cpl_params(cpl)
        self.r_max = float(r_max)
        nb = L.ledds_cpl_workspace_bytes(lbm.h, dem.h, self.c, self.r_max)
        self.cpl_scratch = torch.empty(max(nb, 16), dtype=torch.uint8, device="cuda")
        L.ledds_cpl_init(lbm.h, dem.h, self.c, self.r_max, self.cpl_scratch)
        self.f_hyd = torch.zeros(dem.n, 3, dtype=torch.float64, device="cuda")
        self.m_hyd = torch.zeros(dem.n, 3, dtype=torch.float64, device="cuda")

    def step(self, nsteps=1):
        d = self.dem
        call = L.ledds_coupled_step_f32 if self.lbm.f32 else L.ledds_coupled_step
        call(self.lbm.h, d.h, self.c, self.r_max, self.lbm.f, d.x, d.v, d.w, d.a, d.alpha, d.radius,
             self.f_hyd, self.m_hyd, d.history, d.scratch, self.cpl_scratch, d.status, nsteps)
