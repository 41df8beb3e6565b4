"""Python binding of libledds.so (include/ledds.h): argument marshalling only.

Every step of the LBM / DEM / coupled path runs in the CUDA kernels of csrc/;
PyTorch is used for device memory and streams, nothing else.  There is no CPU
fallback: importing this package without the built library raises.
Function names and argument order follow include/ledds.h.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libledds.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(f"{_LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                      "(paper_2512_04997_b200/build.py); there is no CPU fallback")
_lib = C.CDLL(_LIB_PATH)

LEDDS_OK, LEDDS_EINVAL, LEDDS_EALIGN, LEDDS_ECAPACITY, LEDDS_ECUDA = 0, -1, -2, -3, -4
ST_CONTACT_OVERFLOW, ST_SOLID_OVERFLOW, ST_COINCIDENT, ST_NONFINITE, ST_RADIUS_RANGE, ST_OUT_OF_BOX = 1, 2, 4, 8, 16, 32
EXPORTS = ["ledds_lbm_workspace_bytes", "ledds_lbm_init", "ledds_lbm_import", "ledds_lbm_step", "ledds_lbm_export",
           "ledds_lbm_current", "ledds_lbm_destroy", "ledds_lbm_workspace_bytes_f32", "ledds_lbm_init_f32",
           "ledds_lbm_import_f32", "ledds_lbm_step_f32", "ledds_lbm_export_f32", "ledds_dem_workspace_bytes", "ledds_dem_init", "ledds_dem_step",
           "ledds_dem_query", "ledds_dem_destroy", "ledds_dem_cell_order_static", "ledds_dem_cell_order_static_max_n",
           "ledds_dem_workspace_bytes_f32", "ledds_dem_init_f32", "ledds_dem_step_f32",
           "ledds_dem_query_f32", "ledds_cpl_workspace_bytes", "ledds_cpl_init", "ledds_coupled_step",
           "ledds_coupled_step_f32", "ledds_version",
           "ledds_profile", "ledds_profile_read", "ledds_launch_count"]


class LbmParams(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("tau", C.c_double), ("bc", C.c_int * 3),
                ("u_wall", C.c_double * 18), ("layout", C.c_int), ("variant", C.c_int), ("collision", C.c_int)]


class DemParams(C.Structure):
    _fields_ = [("n", C.c_int), ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("bc", C.c_int * 3),
                ("v_wall", C.c_double * 18), ("cell", C.c_double), ("dt", C.c_double), ("g", C.c_double * 3),
                ("density", C.c_double), ("kn", C.c_double), ("kt", C.c_double), ("restitution", C.c_double),
                ("mu", C.c_double), ("kn_w", C.c_double), ("kt_w", C.c_double), ("restitution_w", C.c_double),
                ("mu_w", C.c_double), ("max_contacts", C.c_int), ("model", C.c_int), ("young", C.c_double),
                ("poisson", C.c_double), ("young_w", C.c_double), ("poisson_w", C.c_double), ("sort_every_step", C.c_int),
                ("no_single_block", C.c_int), ("cell_order", C.c_int)]


class CplParams(C.Structure):
    _fields_ = [("n_sub", C.c_int), ("solid_fraction", C.c_int), ("dx", C.c_double), ("rho_f", C.c_double),
                ("origin", C.c_double * 3)]


class LeddsError(RuntimeError):
    pass


def _check(rc, what):
    if rc != 0:
        name = {-1: "LEDDS_EINVAL", -2: "LEDDS_EALIGN", -3: "LEDDS_ECAPACITY", -4: "LEDDS_ECUDA"}.get(rc, str(rc))
        raise LeddsError(f"{what} failed: {name}")


def _p(t):
    """device pointer of a CUDA tensor (None -> NULL)"""
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda or not t.is_contiguous():
        raise LeddsError("ledds: arguments must be contiguous CUDA tensors")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


for _n in EXPORTS:
    getattr(_lib, _n).restype = C.c_int
_lib.ledds_version.restype = C.c_char_p
_lib.ledds_lbm_current.restype = C.c_void_p
_lib.ledds_launch_count.restype = C.c_ulonglong
K_LBM, K_DEM_KEYS, K_DEM_SORT, K_DEM_GATHER, K_DEM_CONTACT, K_DEM_KICK, K_CPL_REDUCE, K_CPL_RASTER = range(8)
KERNEL_GROUPS = ["lbm", "dem_keys", "dem_sort", "dem_gather", "dem_contact", "dem_kick", "cpl_reduce", "cpl_raster"]


def lbm_params(d) -> LbmParams:
    """dict(shape, tau, bc, u_wall[, variant, collision]) -> ledds_lbm_params"""
    p = LbmParams()
    p.nx, p.ny, p.nz = (int(v) for v in d["shape"])
    p.tau = float(d["tau"])
    p.bc[:] = [int(v) for v in d["bc"]]
    uw = d.get("u_wall")
    p.u_wall[:] = [0.0] * 18 if uw is None else [float(v) for v in list(uw.reshape(-1) if hasattr(uw, "reshape") else uw)]
    p.layout = 0
    p.variant = int(d.get("variant", 0))
    p.collision = int(d.get("collision", 0))
    return p


def dem_params(d) -> DemParams:
    p = DemParams()
    p.n = int(d["n"])
    p.lo[:] = d["lo"]; p.hi[:] = d["hi"]; p.bc[:] = [int(v) for v in d["bc"]]
    vw = d.get("v_wall")
    p.v_wall[:] = [0.0] * 18 if vw is None else [float(v) for v in list(vw.reshape(-1) if hasattr(vw, "reshape") else vw)]
    p.cell = d["cell"]; p.dt = d["dt"]; p.g[:] = d["g"]; p.density = d["density"]
    p.kn = d["kn"]; p.kt = d["kt"]; p.restitution = d["restitution"]; p.mu = d["mu"]
    p.kn_w = d.get("kn_w", d["kn"]); p.kt_w = d.get("kt_w", d["kt"])
    p.restitution_w = d.get("restitution_w", d["restitution"]); p.mu_w = d.get("mu_w", d["mu"])
    p.max_contacts = int(d.get("max_contacts", 16))
    p.model = int(d.get("model", 0))
    p.young = float(d.get("young", 0.0)); p.poisson = float(d.get("poisson", 0.0))
    p.young_w = float(d.get("young_w", p.young)); p.poisson_w = float(d.get("poisson_w", p.poisson))
    p.sort_every_step = int(d.get("sort_every_step", 0))
    p.no_single_block = int(d.get("no_single_block", 0))
    p.cell_order = int(d.get("cell_order", 0))
    return p


def cpl_params(d) -> CplParams:
    p = CplParams()
    p.n_sub = int(d["n_sub"]); p.solid_fraction = int(d.get("solid_fraction", 0))
    p.dx = float(d["dx"]); p.rho_f = float(d["rho_f"])
    p.origin[:] = [float(v) for v in d.get("origin", (0.0, 0.0, 0.0))]
    return p


def ledds_version():
    return _lib.ledds_version().decode()


def ledds_profile(enable: bool):
    _check(_lib.ledds_profile(C.c_int(1 if enable else 0)), "ledds_profile")


def ledds_profile_read(kernel_id: int):
    """-> (total_ms, launches) of one kernel group recorded since ledds_profile(True)"""
    ms, n = C.c_double(0.0), C.c_int(0)
    _check(_lib.ledds_profile_read(C.c_int(kernel_id), C.byref(ms), C.byref(n)), "ledds_profile_read")
    return ms.value, n.value


def ledds_launch_count() -> int:
    return int(_lib.ledds_launch_count())


def ledds_lbm_current(h, f):
    """device address (int) of the current canonical field inside f"""
    return _lib.ledds_lbm_current(h, _p(f))


# ------------------------------------------------------------------------------------ LBM
def ledds_lbm_workspace_bytes(p: LbmParams) -> int:
    n = C.c_size_t(0)
    _check(_lib.ledds_lbm_workspace_bytes(C.byref(p), C.byref(n)), "ledds_lbm_workspace_bytes")
    return n.value


def ledds_lbm_init(p: LbmParams, f, rho=None, u=None):
    h = C.c_void_p(0)
    _check(_lib.ledds_lbm_init(C.byref(h), C.byref(p), _p(f), _p(rho), _p(u), _stream()), "ledds_lbm_init")
    return h


def ledds_lbm_import(h, f, f_canonical):
    _check(_lib.ledds_lbm_import(h, _p(f), _p(f_canonical), _stream()), "ledds_lbm_import")


def ledds_lbm_step(h, f, nsteps=1):
    _check(_lib.ledds_lbm_step(h, _p(f), C.c_int(nsteps), _stream()), "ledds_lbm_step")


def ledds_lbm_export(h, f, f_canonical=None, rho=None, u=None):
    _check(_lib.ledds_lbm_export(h, _p(f), _p(f_canonical), _p(rho), _p(u), _stream()), "ledds_lbm_export")


def ledds_lbm_destroy(h):
    _lib.ledds_lbm_destroy(h)


# fp32 set: same calls on float buffers (include/ledds.h)
def ledds_lbm_workspace_bytes_f32(p: LbmParams) -> int:
    n = C.c_size_t(0)
    _check(_lib.ledds_lbm_workspace_bytes_f32(C.byref(p), C.byref(n)), "ledds_lbm_workspace_bytes_f32")
    return n.value


def ledds_lbm_init_f32(p: LbmParams, f, rho=None, u=None):
    h = C.c_void_p(0)
    _check(_lib.ledds_lbm_init_f32(C.byref(h), C.byref(p), _p(f), _p(rho), _p(u), _stream()), "ledds_lbm_init_f32")
    return h


def ledds_lbm_import_f32(h, f, f_canonical):
    _check(_lib.ledds_lbm_import_f32(h, _p(f), _p(f_canonical), _stream()), "ledds_lbm_import_f32")


def ledds_lbm_step_f32(h, f, nsteps=1):
    _check(_lib.ledds_lbm_step_f32(h, _p(f), C.c_int(nsteps), _stream()), "ledds_lbm_step_f32")


def ledds_lbm_export_f32(h, f, f_canonical=None, rho=None, u=None):
    _check(_lib.ledds_lbm_export_f32(h, _p(f), _p(f_canonical), _p(rho), _p(u), _stream()), "ledds_lbm_export_f32")


# ------------------------------------------------------------------------------------ DEM
def ledds_dem_workspace_bytes(p: DemParams):
    a, b = C.c_size_t(0), C.c_size_t(0)
    _check(_lib.ledds_dem_workspace_bytes(C.byref(p), C.byref(a), C.byref(b)), "ledds_dem_workspace_bytes")
    return a.value, b.value


def ledds_dem_init(p: DemParams, x, v, w, radius, a, alpha, history, scratch, status):
    h = C.c_void_p(0)
    _check(_lib.ledds_dem_init(C.byref(h), C.byref(p), _p(x), _p(v), _p(w), _p(radius), _p(a), _p(alpha), _p(history),
                               _p(scratch), _p(status), _stream()), "ledds_dem_init")
    return h


def ledds_dem_step(h, x, v, w, a, alpha, radius, f_ext, m_ext, history, scratch, status, nsteps=1):
    _check(_lib.ledds_dem_step(h, _p(x), _p(v), _p(w), _p(a), _p(alpha), _p(radius), _p(f_ext), _p(m_ext), _p(history),
                               _p(scratch), _p(status), C.c_int(nsteps), _stream()), "ledds_dem_step")


def ledds_dem_query(h, history, scratch, sorted_idx=None, sorted_key=None, pairs=None, pair_dt=None, pair_cap=0,
                    n_pairs=None, force=None, torque=None):
    _check(_lib.ledds_dem_query(h, _p(history), _p(scratch), _p(sorted_idx), _p(sorted_key), _p(pairs), _p(pair_dt),
                                C.c_uint32(pair_cap), _p(n_pairs), _p(force), _p(torque), _stream()), "ledds_dem_query")


def ledds_dem_destroy(h):
    _lib.ledds_dem_destroy(h)


def ledds_dem_cell_order_static_max_n() -> int:
    return int(_lib.ledds_dem_cell_order_static_max_n())


def ledds_dem_cell_order_static(p: DemParams, x, sorted_idx, sorted_key):
    """(cell key, id) order of the particles at x with the library's static scratch: no workspace, no allocation
    (include/ledds.h).  Calls that overlap on the GPU race."""
    rc = _lib.ledds_dem_cell_order_static(C.byref(p), _p(x), _p(sorted_idx), _p(sorted_key), _stream())
    if rc == -3:
        raise LeddsError(f"ledds_dem_cell_order_static: n = {p.n} particles exceed the static scratch of the library "
                         f"({ledds_dem_cell_order_static_max_n()} particles): LEDDS_ECAPACITY")
    _check(rc, "ledds_dem_cell_order_static")


# fp32 set: same calls on float arrays (include/ledds.h)
def ledds_dem_workspace_bytes_f32(p: DemParams):
    a, b = C.c_size_t(0), C.c_size_t(0)
    _check(_lib.ledds_dem_workspace_bytes_f32(C.byref(p), C.byref(a), C.byref(b)), "ledds_dem_workspace_bytes_f32")
    return a.value, b.value


def ledds_dem_init_f32(p: DemParams, x, v, w, radius, a, alpha, history, scratch, status):
    h = C.c_void_p(0)
    _check(_lib.ledds_dem_init_f32(C.byref(h), C.byref(p), _p(x), _p(v), _p(w), _p(radius), _p(a), _p(alpha), _p(history),
                                   _p(scratch), _p(status), _stream()), "ledds_dem_init_f32")
    return h


def ledds_dem_step_f32(h, x, v, w, a, alpha, radius, f_ext, m_ext, history, scratch, status, nsteps=1):
    _check(_lib.ledds_dem_step_f32(h, _p(x), _p(v), _p(w), _p(a), _p(alpha), _p(radius), _p(f_ext), _p(m_ext), _p(history),
                                   _p(scratch), _p(status), C.c_int(nsteps), _stream()), "ledds_dem_step_f32")


def ledds_dem_query_f32(h, history, scratch, sorted_idx=None, sorted_key=None, pairs=None, pair_dt=None, pair_cap=0,
                        n_pairs=None, force=None, torque=None):
    _check(_lib.ledds_dem_query_f32(h, _p(history), _p(scratch), _p(sorted_idx), _p(sorted_key), _p(pairs), _p(pair_dt),
                                    C.c_uint32(pair_cap), _p(n_pairs), _p(force), _p(torque), _stream()), "ledds_dem_query_f32")


# ------------------------------------------------------------------------------------ coupled
def ledds_cpl_workspace_bytes(lbm, dem, c: CplParams, r_max: float) -> int:
    n = C.c_size_t(0)
    _check(_lib.ledds_cpl_workspace_bytes(lbm, dem, C.byref(c), C.c_double(r_max), C.byref(n)), "ledds_cpl_workspace_bytes")
    return n.value


def ledds_cpl_init(lbm, dem, c: CplParams, r_max: float, cpl_scratch):
    _check(_lib.ledds_cpl_init(lbm, dem, C.byref(c), C.c_double(r_max), _p(cpl_scratch), _stream()), "ledds_cpl_init")


def ledds_coupled_step(lbm, dem, c: CplParams, r_max, f, x, v, w, a, alpha, radius, f_hyd, m_hyd, history, scratch,
                       cpl_scratch, status, nsteps=1):
    _check(_lib.ledds_coupled_step(lbm, dem, C.byref(c), C.c_double(r_max), _p(f), _p(x), _p(v), _p(w), _p(a), _p(alpha),
                                   _p(radius), _p(f_hyd), _p(m_hyd), _p(history), _p(scratch), _p(cpl_scratch),
                                   _p(status), C.c_int(nsteps), _stream()), "ledds_coupled_step")


def ledds_coupled_step_f32(lbm, dem, c: CplParams, r_max, f, x, v, w, a, alpha, radius, f_hyd, m_hyd, history, scratch,
                           cpl_scratch, status, nsteps=1):
    _check(_lib.ledds_coupled_step_f32(lbm, dem, C.byref(c), C.c_double(r_max), _p(f), _p(x), _p(v), _p(w), _p(a), _p(alpha),
                                       _p(radius), _p(f_hyd), _p(m_hyd), _p(history), _p(scratch), _p(cpl_scratch),
                                       _p(status), C.c_int(nsteps), _stream()), "ledds_coupled_step_f32")


from .sim import Lbm, Dem, Coupled  # noqa: E402  (buffer-owning convenience wrappers; no arithmetic)
