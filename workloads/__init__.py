"""Seeded synthetic inputs shaped like BASELINE.json's configs (numpy only).

This module serves BOTH the CPU oracle and the CUDA path and therefore holds
none of the method's arithmetic: it only draws positions, radii, velocities and
fields and fills parameter dicts.  Recipes are stated in DESIGN.md section 4.
The paper's own input decks and experimental curves are not available; these
inputs stand in for its workloads E4 (gas in a box), E6 (ten Cate
settling), E8 (sheared suspension) and E10 (4 M
spheres).
"""
import numpy as np

PI = np.pi


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


# ------------------------------------------------------------------ fluid fields
def tgv(shape, u0=0.02, rho0=1.0, plane="xy"):
    """Two-dimensional Taylor-Green field extruded along the third axis (reading
    G29): u_a = u0 sin(ka a) cos(kb b), u_b = -u0 cos(ka a) sin(kb b) (scaled so it
    stays divergence-free on non-cubic boxes), rho = rho0 [1 + 3 u0^2/4 (cos 2ka a + cos 2kb b)].
    Returns rho [N], u [3, N] with x fastest."""
    nx, ny, nz = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    co = {"x": (x, nx, 0), "y": (y, ny, 1), "z": (z, nz, 2)}
    (a, na, ia), (b, nb, ib) = co[plane[0]], co[plane[1]]
    ka, kb = 2 * PI / na, 2 * PI / nb
    u = np.zeros((3,) + x.shape)
    u[ia] = u0 * np.sin(ka * a) * np.cos(kb * b)
    u[ib] = -u0 * (ka / kb) * np.cos(ka * a) * np.sin(kb * b)
    rho = rho0 * (1.0 + 0.75 * u0 * u0 * (np.cos(2 * ka * a) + np.cos(2 * kb * b)))
    return rho.reshape(-1), u.reshape(3, -1)


def random_flow(shape, seed, amp=0.02):
    """Smooth-free random rho, u (white noise of small amplitude) for parity tests."""
    n = shape[0] * shape[1] * shape[2]
    g = _rng(seed)
    return 1.0 + 0.01 * g.standard_normal(n), amp * g.standard_normal((3, n))


# ------------------------------------------------------------------ particles
def rsa(seed, n, lo, hi, radius, periodic=(False, False, False), batch=20000, max_batches=4000):
    """Random sequential addition of n non-overlapping spheres with centres in
    [lo, hi] (closed box for the centres).  radius: array of n radii, placed in
    the given order.  Returns x [n,3] (or raises if the box is too full)."""
    g = _rng(seed)
    lo = np.asarray(lo, float); hi = np.asarray(hi, float)
    radius = np.asarray(radius, float)
    L = hi - lo
    per = np.asarray(periodic, bool)
    h = 2.0 * radius.max()
    nc = np.maximum(1, np.floor(L / h).astype(int))
    nc = np.where(per & (nc < 3), 1, nc)
    K = 8
    members = -np.ones((nc[0] * nc[1] * nc[2], K), np.int64)
    count = np.zeros(nc[0] * nc[1] * nc[2], np.int64)
    x = np.zeros((n, 3))
    offs = np.array([(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)])

    def cells_of(p):
        c = np.floor((p - lo) / L * nc).astype(int)
        return np.clip(c, 0, nc - 1)

    def neighbours(c):
        q = c[:, None, :] + offs[None, :, :]
        ok = np.ones(q.shape[:2], bool)
        for a in range(3):
            if per[a]:
                q[..., a] %= nc[a]
            else:
                ok &= (q[..., a] >= 0) & (q[..., a] < nc[a])
                q[..., a] = np.clip(q[..., a], 0, nc[a] - 1)
        return q[..., 0] + nc[0] * (q[..., 1] + nc[1] * q[..., 2]), ok

    def overlaps(p, rp, placed):
        """p [m,3], rp [m] -> bool [m]: overlaps any sphere already in the grid."""
        lin, ok = neighbours(cells_of(p))
        mem = members[lin]                                   # [m, 27, K]
        valid = (mem >= 0) & ok[..., None]
        mem = np.where(valid, mem, 0)
        dist2 = np.zeros(mem.shape)
        for a in range(3):
            d = p[:, a][:, None, None] - x[:, a][mem]
            if per[a]:
                d -= L[a] * np.round(d / L[a])
            dist2 += d * d
        rr = rp[:, None, None] + radius[mem]
        return (valid & (dist2 < rr * rr)).any(axis=(1, 2))

    placed = 0
    for _ in range(max_batches):
        if placed >= n:
            break
        m = min(batch, max(4 * (n - placed), 256))
        cand = lo + g.random((m, 3)) * L
        # candidates are offered to the next unplaced spheres in order; a rejected one is dropped
        keep = np.nonzero(~overlaps(cand, np.full(m, radius[placed:].max()), placed))[0] if placed else np.arange(m)
        for ci in keep:
            if placed >= n:
                break
            p = cand[ci:ci + 1]
            if overlaps(p, radius[placed:placed + 1], placed)[0]:
                continue
            x[placed] = p[0]
            c = cells_of(p)[0]
            lin = c[0] + nc[0] * (c[1] + nc[1] * c[2])
            if count[lin] >= K:
                raise RuntimeError("rsa: cell capacity exceeded")
            members[lin, count[lin]] = placed
            count[lin] += 1
            placed += 1
    if placed < n:
        raise RuntimeError(f"rsa: placed only {placed} of {n}")
    return x


def dem_defaults(n, lo, hi, bc, cell, dt, g, density, kn, restitution, mu, kt=None, **kw):
    d = dict(n=int(n), lo=tuple(map(float, lo)), hi=tuple(map(float, hi)), bc=tuple(bc), cell=float(cell), dt=float(dt),
             g=tuple(map(float, g)), density=float(density), kn=float(kn), kt=float(kn * 2.0 / 7.0 if kt is None else kt),
             restitution=float(restitution), mu=float(mu), v_wall=np.zeros(18))
    d.update(kw)
    d.setdefault("kn_w", d["kn"]); d.setdefault("kt_w", d["kt"])
    d.setdefault("restitution_w", d["restitution"]); d.setdefault("mu_w", d["mu"])
    d.setdefault("max_contacts", 16)
    return d


# ------------------------------------------------------------------ BASELINE configs
def cfg1_gas(seed=1, sites=(16, 16, 8)):
    """configs[0]: DEM-only gas of monodisperse spheres in a closed box (reading G30)."""
    R, d = 0.5e-3, 1.0e-3
    sp = 1.02 * d
    sx, sy, sz = sites
    n = sx * sy * sz
    g = _rng(seed)
    k, j, i = np.meshgrid(np.arange(sz), np.arange(sy), np.arange(sx), indexing="ij")
    x = np.stack([(i + 0.5) * sp, (j + 0.5) * sp, (k + 0.5) * sp], -1).reshape(n, 3)
    x = x + g.uniform(-0.05 * d, 0.05 * d, (n, 3))
    v = g.normal(0.0, 0.05, (n, 3))
    pd = dem_defaults(n, (0, 0, 0), (sx * sp, sy * sp, sz * sp), (1, 1, 1), cell=d, dt=1e-6, g=(0, 0, -9.81),
                      density=2500.0, kn=1e4, restitution=0.7, mu=0.3)
    return pd, x, v, np.zeros((n, 3)), np.full(n, R)


def cfg2_tgv(n=128):
    """configs[1]: LBM-only periodic Taylor-Green vortex."""
    shape = (n, n, n)
    rho, u = tgv(shape, 0.02, 1.0, "xy")
    return dict(shape=shape, tau=0.6, bc=(0, 0, 0), u_wall=np.zeros(18)), rho, u


def cfg3_settling(shape=(64, 64, 256), R=6.0, z0=200.0, g=1.0e-4):
    """configs[2]: one sphere settling in a closed box of quiescent fluid (G31).
    Lattice units for everything (dx = 1, rho_f = 1, dt = 1, n_sub = 1); lattice node
    i sits at coordinate i, the walls at -1/2 and n-1/2 (G19)."""
    nx, ny, nz = shape
    ratio = 1.5
    lbm = dict(shape=shape, tau=0.55, bc=(1, 1, 1), u_wall=np.zeros(18))
    cpl = dict(n_sub=1, dx=1.0, rho_f=1.0, origin=(0.0, 0.0, 0.0))
    geff = -(1.0 - 1.0 / ratio) * g                       # Eq. (56), computed by the harness
    pd = dem_defaults(1, (-0.5, -0.5, -0.5), (nx - 0.5, ny - 0.5, nz - 0.5), (1, 1, 1), cell=2 * R + 2.0, dt=1.0,
                      g=(0, 0, geff), density=ratio, kn=5.36, restitution=0.7, mu=0.3)
    x = np.array([[nx / 2.0, ny / 2.0, z0]])
    return lbm, cpl, pd, x, np.zeros((1, 3)), np.zeros((1, 3)), np.full(1, R)


def cfg4_shear(seed=4, n=256, n_part=20000, R=4.0, uw=0.05):
    """configs[3]: neutrally buoyant spheres in plane Couette flow, periodic x,y,
    walls z moving at u_x = -/+ uw.  RSA placement, initial v = local Couette velocity."""
    shape = (n, n, n)
    u_wall = np.zeros((3, 2, 3))
    u_wall[2, 0, 0] = -uw
    u_wall[2, 1, 0] = +uw
    lbm = dict(shape=shape, tau=0.6, bc=(0, 0, 1), u_wall=u_wall.reshape(-1))
    cpl = dict(n_sub=1, dx=1.0, rho_f=1.0, origin=(0.0, 0.0, 0.0))
    lo, hi = (-0.5, -0.5, -0.5), (n - 0.5, n - 0.5, n - 0.5)
    radius = np.full(n_part, R)
    x = rsa(seed, n_part, (lo[0], lo[1], R - 0.5), (hi[0], hi[1], n - 0.5 - R), radius, periodic=(True, True, False))
    m = (4.0 / 3.0) * PI * R ** 3
    kn = 0.5 * m * (PI / 50.0) ** 2                       # m* = m/2; contact lasts ~50 dt (G31)
    pd = dem_defaults(n_part, lo, hi, (0, 0, 1), cell=2 * R + 1.3, dt=1.0, g=(0, 0, 0), density=1.0, kn=kn,
                      restitution=0.95, mu=0.3, v_wall=u_wall.reshape(-1))
    v = np.zeros((n_part, 3))
    v[:, 0] = -uw + 2 * uw * (x[:, 2] + 0.5) / n
    # fluid starts from the Couette profile as well
    zz = np.repeat(np.arange(n), n * n)
    u = np.zeros((3, n ** 3))
    u[0] = -uw + 2 * uw * (zz + 0.5) / n
    return lbm, cpl, pd, x, v, np.zeros((n_part, 3)), radius, u


def cfg5_pour(seed=5, n_side=160, n_part=4_000_000, dense=False):
    """configs[4]: polydisperse spheres, R ~ U(0.8, 1.2) r0, in the upper half of a
    (2.5 n_side r0)^2 x (5 n_side r0) walled box (400 x 400 x 800 r0 at n_side = 160).
    Placement = the documented fallback to RSA: seeded jittered cubic lattice at
    spacing 2.5 r0 (no overlaps).  dense=True is the supplementary dense state:
    spacing 2.0 r0 at the bottom of the box, radii anti-correlated on a
    checkerboard so that about half the lattice neighbours overlap slightly."""
    r0 = 1.0e-3
    g = _rng(seed)
    box = (2.5 * n_side * r0, 2.5 * n_side * r0, 5.0 * n_side * r0)
    n_part = min(n_part, n_side ** 3)
    sites = g.permutation(n_side ** 3)[:n_part]
    i, j, k = sites % n_side, (sites // n_side) % n_side, sites // (n_side * n_side)
    if not dense:
        sp = 2.5 * r0
        radius = r0 * g.uniform(0.8, 1.2, n_part)
        x = np.stack([(i + 0.5) * sp, (j + 0.5) * sp, (k + 0.5) * sp + 0.5 * box[2]], -1)
        x += g.uniform(-0.04 * r0, 0.04 * r0, (n_part, 3))
    else:
        sp = 2.0 * r0
        sign = np.where((i + j + k) % 2 == 0, 1.0, -1.0)
        radius = r0 * (1.0 + 0.2 * sign * g.uniform(0.0, 1.0, n_part))
        x = np.stack([(i + 0.5) * sp, (j + 0.5) * sp, (k + 0.5) * sp], -1) + 0.6 * r0
        x += g.uniform(-0.01 * r0, 0.01 * r0, (n_part, 3))
    pd = dem_defaults(n_part, (0, 0, 0), box, (1, 1, 1), cell=2.4 * r0, dt=2e-6, g=(0, 0, -9.81), density=2500.0,
                      kn=1e4, restitution=0.5, mu=0.5, max_contacts=16)
    return pd, x, np.zeros((n_part, 3)), np.zeros((n_part, 3)), radius


def dem_random(seed, n, box=(10.0, 10.0, 10.0), bc=(1, 1, 1), rmin=0.4, rmax=0.6, overlap=True):
    """Small random DEM state with overlapping polydisperse spheres (parity / pin tests)."""
    g = _rng(seed)
    x = g.random((n, 3)) * np.asarray(box)
    radius = g.uniform(rmin, rmax, n)
    v = g.normal(0.0, 1.0, (n, 3)); w = g.normal(0.0, 1.0, (n, 3))
    pd = dem_defaults(n, (0, 0, 0), box, bc, cell=2 * rmax, dt=1e-4, g=(0, 0, -9.81), density=1000.0, kn=1e5,
                      restitution=0.8, mu=0.4)
    return pd, x, v, w, radius


def paper_bed(phi, shape=(500, 200, 800), D=20.0, seed=6, n_sub=10, contacts=False):
    """the paper's performance workload: a 500 x 200 x 800 lattice,
    spheres of diameter 20 cells at solid fraction phi (0 / 0.15 / 0.30 / 0.45 -> 0 / 2 866 / 5 731 / 8 596 spheres
    in the paper), density ratio 1.1, 10 DEM sub-steps per LBM step, TRT collision.  The paper's inlet / outlet
    are not part of the hot path: here the box is periodic in x, y with walls in z, fluid at rest, gravity on
    the spheres.  Placement: seeded jittered simple-cubic lattice at the spacing that gives phi (RSA cannot
    reach 0.45), filled from the bottom.  contacts=True: the same number of spheres stacked in vertical columns
    whose neighbours overlap by 0.4 % of a diameter (the lowest one rests on the floor), so that the bed has
    about one contact per sphere from the first step on and the DEM contact path is loaded."""
    nx, ny, nz = shape
    R = 0.5 * D
    lbm = dict(shape=shape, tau=0.6, bc=(0, 0, 1), u_wall=np.zeros(18), collision=1)
    cpl = dict(n_sub=n_sub, dx=1.0, rho_f=1.0, origin=(0.0, 0.0, 0.0))
    lo, hi = (-0.5, -0.5, -0.5), (nx - 0.5, ny - 0.5, nz - 0.5)
    vol = (4.0 / 3.0) * PI * R ** 3
    n_part = int(round(phi * nx * ny * nz / vol))
    g = _rng(seed)
    if n_part > 0 and contacts:
        szc = 2.0 * R * 0.996
        best = None
        for mx in range(max(1, int(nx // (2 * R)) - 8), int(nx // (2 * R)) + 1):
            for my in range(max(1, int(ny // (2 * R)) - 4), int(ny // (2 * R)) + 1):
                sx, sy = nx / mx, ny / my
                layers = -(-n_part // (mx * my))
                if min(sx, sy) <= 2.0 * R + 0.2 or layers * szc + 2.0 > nz:
                    continue
                if best is None or min(sx, sy) > best[0]:
                    best = (min(sx, sy), mx, my, sx, sy)
        assert best is not None, "bed does not fit at this fraction"
        _, mx, my, sx, sy = best
        sites = np.arange(n_part)
        i, j, k = sites % mx, (sites // mx) % my, sites // (mx * my)
        x = np.stack([(i + 0.5) * sx - 0.5, (j + 0.5) * sy - 0.5, -0.5 + 0.996 * R + k * szc], -1)
        x[:, :2] += g.uniform(-0.05, 0.05, (n_part, 2))
        x = x[g.permutation(n_part)]
    elif n_part > 0:
        # lattice spacing for the target fraction, snapped so that whole cells fit the periodic directions
        s = (vol / phi) ** (1.0 / 3.0)
        best = None
        for mx in (int(nx // s), int(nx // s) + 1):
            for my in (int(ny // s), int(ny // s) + 1):
                sx, sy = nx / mx, ny / my
                sz = vol / (phi * sx * sy)
                if best is None or min(sx, sy, sz) > best[0]:
                    best = (min(sx, sy, sz), mx, my, sx, sy, sz)
        _, mx, my, sx, sy, sz = best
        mz = int((nz - 1.0) // sz)
        n_part = min(n_part, mx * my * mz)
        sites = np.arange(mx * my * mz)[:n_part]
        i, j, k = sites % mx, (sites // mx) % my, sites // (mx * my)
        x = np.stack([(i + 0.5) * sx - 0.5, (j + 0.5) * sy - 0.5, (k + 0.5) * sz], -1)
        slack = 0.5 * (min(sx, sy, sz) - 2.0 * R)
        assert slack > 0.0, "spheres would overlap at this fraction"
        x = x + g.uniform(-0.4 * slack, 0.4 * slack, (n_part, 3))
        x = x[g.permutation(n_part)]
    else:
        x = np.zeros((0, 3))
    m = 1.1 * vol
    kn = 0.5 * m * (PI / (50.0 / n_sub)) ** 2               # contact lasts ~50 DEM steps (dt = 1/n_sub)
    pd = dem_defaults(n_part, lo, hi, (0, 0, 1), cell=2 * R + 1.3, dt=1.0 / n_sub, g=(0, 0, -(1.0 - 1.0 / 1.1) * 1e-5),
                      density=1.1, kn=kn, restitution=0.9, mu=0.3)
    return lbm, cpl, pd, x, np.zeros((n_part, 3)), np.zeros((n_part, 3)), np.full(n_part, R)
