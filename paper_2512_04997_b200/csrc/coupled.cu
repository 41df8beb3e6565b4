// Fluid-solid coupling through partially saturated cells (PSM), Eq. (32)-(42),
// fused into the D3Q19 stream-collide pass, plus the coupled step driver.
//
//   lbm_psm_kernel     per fluid cell: find the (<= 2, lowest ids) solids cutting it in the 2x2x2
//                      DEM grid cells around it (sorted particle arrays of the DEM pass), solid
//                      fraction Eq. (39)-(40), weights Eq. (36)-(37), PSM collision Eq. (32)-(35),
//                      streaming with boundaries; the per-(cell, solid) momentum exchange of
//                      Eq. (41)-(42) is written to that solid's private box of partials.
//   cpl_reduce_kernel  one block per solid: deterministic sum of its box -> F_sf, M_sf (no atomics,
//                      no sort over N_fluid as in PAPER.md:525-530).
#include <math.h>

#include "lbm_kernels.cuh"

struct CplDev {
    int n;
    double rc;                 // Eq. (40) in lattice units
    double inv_dx, vscale, wscale, origin[3];
    double fscale, mscale;     // lattice -> DEM units for force / torque
    // DEM grid seen from lattice indices: grid coordinate = r * gs + g0, search half-width dg
    int nc[3], gbc[3];
    double gs[3], g0[3], dg[3];
    int H, S;                  // box of partials per solid: S^3 entries of 6 doubles
    const uint32_t* cell_start; const uint32_t* cell_end; const uint32_t* sidx;
    const double* xs; const double* vps; const double* wps; const double* rs;
    double* boxes;
    int32_t* status;
};

// delta_sc of Eq. (40) > 0, evaluated with explicitly rounded operations so that the collide kernel
// and the reduce kernel take the same decision for the same (cell, solid).
__device__ __forceinline__ double cpl_dist(const double* d)
{
    return __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
}
__device__ __forceinline__ double cpl_dsc(double Rk, double rc, double dist) { return __dsub_rn(__dadd_rn(Rk, rc), dist); }

// lattice node image nearest to the solid: integer offset di = r - floor(xk), wrapped on periodic axes
__device__ __forceinline__ int cpl_offset(int r, int fk, int n, int periodic)
{
    int di = r - fk;
    if (periodic) {
        if (2 * di > n) di -= n;
        else if (2 * di < -n) di += n;
    }
    return di;
}

__global__ void __launch_bounds__(128) lbm_psm_kernel(const double* __restrict__ fin, double* __restrict__ fout,
                                                      const LbmDev P, const CplDev C)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= P.nx) return;
    const long long cell = ((long long)z * P.ny + y) * P.nx + x;
    double f[LEDDS_Q];
#pragma unroll
    for (int q = 0; q < LEDDS_Q; ++q) f[q] = __ldg(fin + (long long)q * P.N + cell);

    // ---- which solids cut this cell (two lowest ids with beta > 0) ----
    const int r[3] = {x, y, z};
    const int nl[3] = {P.nx, P.ny, P.nz};
    int clo[3], chi[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double g = r[a] * C.gs[a] + C.g0[a];
        clo[a] = (int)floor(g - C.dg[a]);
        chi[a] = (int)floor(g + C.dg[a]);
        if (C.gbc[a]) { clo[a] = max(clo[a], 0); chi[a] = min(chi[a], C.nc[a] - 1); }
    }
    uint32_t id0 = 0xffffffffu, id1 = 0xffffffffu, t0 = 0, t1 = 0;
    int extra = 0;
    for (int gz = clo[2]; gz <= chi[2]; ++gz) {
        const int wz = C.gbc[2] ? gz : (gz % C.nc[2] + C.nc[2]) % C.nc[2];
        for (int gy = clo[1]; gy <= chi[1]; ++gy) {
            const int wy = C.gbc[1] ? gy : (gy % C.nc[1] + C.nc[1]) % C.nc[1];
            for (int gx = clo[0]; gx <= chi[0]; ++gx) {
                const int wx = C.gbc[0] ? gx : (gx % C.nc[0] + C.nc[0]) % C.nc[0];
                const uint32_t gc = (uint32_t)(wx + C.nc[0] * (wy + C.nc[1] * wz));
                const uint32_t b = C.cell_start[gc], e = C.cell_end[gc];
                for (uint32_t t = b; t < e; ++t) {
                    double d[3];
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        const double xk = (C.xs[3 * t + a] - C.origin[a]) * C.inv_dx;
                        const int fk = (int)floor(xk);
                        d[a] = (double)(fk + cpl_offset(r[a], fk, nl[a], !P.bc[a])) - xk;
                    }
                    if (!(cpl_dsc(C.rs[t] * C.inv_dx, C.rc, cpl_dist(d)) > 0.0)) continue;
                    const uint32_t id = C.sidx[t];
                    if (id == id0 || id == id1) continue;                  // same solid seen through a wrapped cell
                    if (id < id0) { if (id1 != 0xffffffffu) ++extra; id1 = id0; t1 = t0; id0 = id; t0 = t; }
                    else if (id < id1) { if (id1 != 0xffffffffu) ++extra; id1 = id; t1 = t; }
                    else ++extra;
                }
            }
        }
    }

    double rho, ux, uy, uz;
    lb_moments(f, rho, ux, uy, uz);
    if (id0 == 0xffffffffu) {
        lb_collide_bgk(f, P.omega, rho, ux, uy, uz);                         // plain collide-and-stream
    } else {
        if (extra) {
            // more than two solids (PAPER.md:515 allows two): flag it and give every dropped solid a
            // zero partial so that its reduction never reads a stale entry
            atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
            for (int gz = clo[2]; gz <= chi[2]; ++gz)
                for (int gy = clo[1]; gy <= chi[1]; ++gy)
                    for (int gx = clo[0]; gx <= chi[0]; ++gx) {
                        const int wz = C.gbc[2] ? gz : (gz % C.nc[2] + C.nc[2]) % C.nc[2];
                        const int wy = C.gbc[1] ? gy : (gy % C.nc[1] + C.nc[1]) % C.nc[1];
                        const int wx = C.gbc[0] ? gx : (gx % C.nc[0] + C.nc[0]) % C.nc[0];
                        const uint32_t gc = (uint32_t)(wx + C.nc[0] * (wy + C.nc[1] * wz));
                        for (uint32_t t = C.cell_start[gc]; t < C.cell_end[gc]; ++t) {
                            const uint32_t id = C.sidx[t];
                            if (id == id0 || id == id1) continue;
                            double d[3];
                            int loc[3];
                            for (int a = 0; a < 3; ++a) {
                                const double xk = (C.xs[3 * t + a] - C.origin[a]) * C.inv_dx;
                                const int fk = (int)floor(xk);
                                const int di = cpl_offset(r[a], fk, nl[a], !P.bc[a]);
                                d[a] = (double)(fk + di) - xk;
                                loc[a] = di + C.H;
                            }
                            if (!(cpl_dsc(C.rs[t] * C.inv_dx, C.rc, cpl_dist(d)) > 0.0)) continue;
                            double* e = C.boxes + (((long long)id * C.S + loc[2]) * C.S + loc[1]) * C.S * 6 + (long long)loc[0] * 6;
                            for (int c = 0; c < 6; ++c) e[c] = 0.0;
                        }
                    }
        }
        double fe[LEDDS_Q], solid[LEDDS_Q];
        lb_equilibrium(fe, rho, ux, uy, uz);
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) solid[q] = 0.0;
        double Bsum = 0.0;
        const int ns = id1 == 0xffffffffu ? 1 : 2;
        for (int s = 0; s < ns; ++s) {
            const uint32_t t = s ? t1 : t0, id = s ? id1 : id0;
            double d[3], xk[3];
            int loc[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                xk[a] = (C.xs[3 * t + a] - C.origin[a]) * C.inv_dx;
                const int fk = (int)floor(xk[a]);
                const int di = cpl_offset(r[a], fk, nl[a], !P.bc[a]);
                d[a] = (double)(fk + di) - xk[a];
                loc[a] = di + C.H;
            }
            const double Rk = C.rs[t] * C.inv_dx;
            const double dsc = cpl_dsc(Rk, C.rc, cpl_dist(d));
            const double beta = dsc >= 2.0 * C.rc ? 1.0 : dsc / (2.0 * C.rc);           // Eq. (39)
            const double B = beta * (P.tau - 0.5) / ((1.0 - beta) + (P.tau - 0.5));     // Eq. (36)
            const double vk[3] = {C.vps[3 * t] * C.vscale, C.vps[3 * t + 1] * C.vscale, C.vps[3 * t + 2] * C.vscale};
            const double wk[3] = {C.wps[3 * t] * C.wscale, C.wps[3 * t + 1] * C.wscale, C.wps[3 * t + 2] * C.wscale};
            const double ukx = vk[0] + (wk[1] * d[2] - wk[2] * d[1]);                   // Eq. (35)
            const double uky = vk[1] + (wk[2] * d[0] - wk[0] * d[2]);
            const double ukz = vk[2] + (wk[0] * d[1] - wk[1] * d[0]);
            double fk_eq[LEDDS_Q];
            lb_equilibrium(fk_eq, rho, ukx, uky, ukz);
            double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma unroll
            for (int q = 0; q < LEDDS_Q; ++q) {
                const int o = lb_opp(q);
                const double Os = (f[o] - fe[o]) - (f[q] - fk_eq[q]);                   // Eq. (34)
                if (lb_cx(q) == 1) sx += Os; else if (lb_cx(q) == -1) sx -= Os;
                if (lb_cy(q) == 1) sy += Os; else if (lb_cy(q) == -1) sy -= Os;
                if (lb_cz(q) == 1) sz += Os; else if (lb_cz(q) == -1) sz -= Os;
                solid[q] += B * Os;
            }
            Bsum += B;
            const double dF[3] = {-B * sx, -B * sy, -B * sz};                           // Eq. (41), lattice units
            double* e = C.boxes + (((long long)id * C.S + loc[2]) * C.S + loc[1]) * C.S * 6 + (long long)loc[0] * 6;
            e[0] = dF[0]; e[1] = dF[1]; e[2] = dF[2];
            e[3] = d[1] * dF[2] - d[2] * dF[1];                                         // Eq. (42)
            e[4] = d[2] * dF[0] - d[0] * dF[2];
            e[5] = d[0] * dF[1] - d[1] * dF[0];
        }
        const double Btot = Bsum < 1.0 ? Bsum : 1.0;                                    // Eq. (37)
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) {
            const double bgk = -P.omega * (f[q] - fe[q]);
            f[q] = f[q] + ((1.0 - Btot) * bgk + solid[q]);                              // Eq. (32)-(33)
        }
    }
    lb_push_store(fout, P, x, y, z, f, rho);
}

// One block per solid: sum the partials of the cells it cuts (same predicate as the collide kernel),
// fixed thread->entry map and fixed tree, so the result is deterministic.
__global__ void __launch_bounds__(256) cpl_reduce_kernel(const LbmDev P, const CplDev C,
                                                         const double* __restrict__ x, const double* __restrict__ radius,
                                                         double* __restrict__ f_hyd, double* __restrict__ m_hyd)
{
    const int k = blockIdx.x;
    const int nl[3] = {P.nx, P.ny, P.nz};
    double xk[3];
    int fk[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        xk[a] = (x[3 * k + a] - C.origin[a]) * C.inv_dx;
        fk[a] = (int)floor(xk[a]);
    }
    const double Rk = radius[k] * C.inv_dx;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    const int S = C.S, S3 = S * S * S;
    const double* box = C.boxes + (long long)k * S3 * 6;
    for (int e = threadIdx.x; e < S3; e += blockDim.x) {
        const int l[3] = {e % S, (e / S) % S, e / (S * S)};
        double d[3];
        bool ok = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int ri = fk[a] + (l[a] - C.H);
            if (P.bc[a] && (ri < 0 || ri >= nl[a])) ok = false;             // outside a walled lattice
            d[a] = (double)ri - xk[a];
        }
        if (!ok) continue;
        if (!(cpl_dsc(Rk, C.rc, cpl_dist(d)) > 0.0)) continue;
#pragma unroll
        for (int c = 0; c < 6; ++c) acc[c] += box[(long long)e * 6 + c];
    }
    __shared__ double red[6][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        double v = acc[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[c][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double v = 0.0;
        for (int w2 = 0; w2 < (int)(blockDim.x >> 5); ++w2) v += red[threadIdx.x][w2];
        if (threadIdx.x < 3) f_hyd[3 * k + threadIdx.x] = v * C.fscale;
        else m_hyd[3 * k + threadIdx.x - 3] = v * C.mscale;
    }
}

// ------------------------------------------------------------------------------------ host API
static int cpl_setup(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c, double r_max, CplDev* C)
{
    if (!lbm || !dem || !c || c->n_sub < 1 || c->solid_fraction != 0 || !(c->dx > 0.0) || !(c->rho_f > 0.0) || !(r_max > 0.0))
        return LEDDS_EINVAL;
    const double rc = cbrt(3.0 / (4.0 * 3.14159265358979323846));
    const double Dt = c->n_sub * dem->d.dt;
    C->n = dem->d.n;
    C->rc = rc;
    C->inv_dx = 1.0 / c->dx;          // positions are divided by dx through this reciprocal only when dx == 1 is exact
    C->vscale = Dt / c->dx;
    C->wscale = Dt;
    C->fscale = c->rho_f * pow(c->dx, 4) / (Dt * Dt);
    C->mscale = c->rho_f * pow(c->dx, 5) / (Dt * Dt);
    const double reach = r_max + rc * c->dx;                                // DEM units
    const int nl[3] = {lbm->d.nx, lbm->d.ny, lbm->d.nz};
    C->H = (int)ceil(r_max / c->dx + rc);
    C->S = 2 * C->H + 2;
    for (int a = 0; a < 3; ++a) {
        C->origin[a] = c->origin[a];
        C->nc[a] = dem->d.nc[a];
        C->gbc[a] = dem->d.bc[a];
        if (dem->d.bc[a] != lbm->d.bc[a]) return LEDDS_EINVAL;              // same topology on both grids
        const double h = dem->d.L[a] / dem->d.nc[a];
        if (dem->d.nc[a] > 1 && h < 2.0 * reach) return LEDDS_EINVAL;       // solids must be found in 2x2x2 grid cells
        C->gs[a] = c->dx * dem->d.inv_h[a];
        C->g0[a] = (c->origin[a] - dem->d.lo[a]) * dem->d.inv_h[a];
        C->dg[a] = reach * dem->d.inv_h[a] * (1.0 + 1e-9) + 1e-9;
        if (!lbm->d.bc[a] && nl[a] < 2 * C->S) return LEDDS_EINVAL;         // unambiguous nearest image
    }
    return LEDDS_OK;
}

extern "C" int ledds_cpl_workspace_bytes(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c,
                                         const double r_max, size_t* bytes)
{
    CplDev C;
    const int rc = cpl_setup(lbm, dem, c, r_max, &C);
    if (rc) return rc;
    if (!bytes) return LEDDS_EINVAL;
    *bytes = (size_t)C.n * C.S * C.S * C.S * 6 * sizeof(double);
    return LEDDS_OK;
}

extern "C" int ledds_coupled_step(ledds_lbm* lbm, ledds_dem* dem, const ledds_cpl_params* c, double r_max, double* f,
                                  double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                                  double* f_hyd, double* m_hyd, void* history, void* scratch, void* cpl_scratch,
                                  int32_t* status, int nsteps, void* stream)
{
    if (!f || !x || !v || !w || !a || !alpha || !radius || !f_hyd || !m_hyd || !history || !scratch || !cpl_scratch ||
        !status || nsteps < 0)
        return LEDDS_EINVAL;
    const void* ptrs[] = {f, x, v, w, a, alpha, radius, f_hyd, m_hyd, history, scratch, cpl_scratch, status};
    for (const void* q : ptrs)
        if (!ledds_aligned16(q)) return LEDDS_EALIGN;
    CplDev C;
    int rc = cpl_setup(lbm, dem, c, r_max, &C);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const DemScratch& s = dem->s;
    char* sc = static_cast<char*>(scratch);
    C.cell_start = reinterpret_cast<const uint32_t*>(sc + s.cell_start);
    C.cell_end = reinterpret_cast<const uint32_t*>(sc + s.cell_end);
    C.xs = reinterpret_cast<const double*>(sc + s.xs);
    C.vps = reinterpret_cast<const double*>(sc + s.vps);
    C.wps = reinterpret_cast<const double*>(sc + s.wps);
    C.rs = reinterpret_cast<const double*>(sc + s.rs);
    C.boxes = static_cast<double*>(cpl_scratch);
    C.status = status;
    const LbmDev& d = lbm->d;
    const size_t half = (size_t)LEDDS_Q * d.N;
    if (d.ny > 65535 || d.nz > 65535) return LEDDS_EINVAL;
    for (int step = 0; step < nsteps; ++step) {
        for (int sub = 0; sub < c->n_sub; ++sub) {
            rc = ledds_dem_advance_contacts(dem, x, v, w, a, alpha, radius, history, scratch, status, dem->d.dt, true, st);
            if (rc) return rc;
            if (sub < c->n_sub - 1) {                                        // F_sf of the previous LBM step is held
                rc = ledds_dem_kick(dem, v, w, a, alpha, radius, f_hyd, m_hyd, scratch, status, st);
                if (rc) return rc;
                dem->steps++;
            }
        }
        C.sidx = reinterpret_cast<const uint32_t*>(sc + s.idx[dem->sorted_buf]);
        dim3 block(128), grid((d.nx + 127) / 128, d.ny, d.nz);
        ledds_prof_start(LEDDS_K_LBM, st);
        lbm_psm_kernel<<<grid, block, 0, st>>>(f + lbm->parity * half, f + (1 - lbm->parity) * half, d, C);
        ledds_prof_stop(LEDDS_K_LBM, st);
        LEDDS_CHECK_LAUNCH();
        lbm->parity ^= 1;
        lbm->steps++;
        ledds_prof_start(LEDDS_K_CPL_REDUCE, st);
        cpl_reduce_kernel<<<C.n, 256, 0, st>>>(d, C, x, radius, f_hyd, m_hyd);
        ledds_prof_stop(LEDDS_K_CPL_REDUCE, st);
        LEDDS_CHECK_LAUNCH();
        rc = ledds_dem_kick(dem, v, w, a, alpha, radius, f_hyd, m_hyd, scratch, status, st);
        if (rc) return rc;
        dem->steps++;
    }
    return LEDDS_OK;
}
