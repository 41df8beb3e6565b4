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

#include "psm_kernels.cuh"

// Cold path: the block's shared candidate list overflowed (never at resolved-particle densities), so the
// thread searches the 2x2x2 DEM grid cells around its own cell in global memory.
__device__ __noinline__ void psm_cell_global_search(const LbmDev& P, const CplDev& C, const int* r, double (&f)[LEDDS_Q],
                                                    double rho, double ux, double uy, double uz)
{
    int clo[3], chi[3];
    for (int a = 0; a < 3; ++a) {
        const double g = r[a] * C.gs[a] + C.g0[a];
        clo[a] = (int)floor(g - C.dg[a]); chi[a] = (int)floor(g + C.dg[a]);
        if (C.gbc[a]) { clo[a] = max(clo[a], 0); chi[a] = min(chi[a], C.nc[a] - 1); }
    }
    uint32_t id0 = 0xffffffffu, id1 = 0xffffffffu;
    int c0 = 0, c1 = 0;
    bool dropped = false;
    PsmCand far0, far1;
    for (int pass = 0; pass < 2; ++pass) {                       // pass 0: select; pass 1: zero the dropped ones
        if (pass == 1 && !dropped) break;
        for (int gz = clo[2]; gz <= chi[2]; ++gz)
            for (int gy = clo[1]; gy <= chi[1]; ++gy)
                for (int gx = clo[0]; gx <= chi[0]; ++gx) {
                    const int wz = C.gbc[2] ? gz : (gz % C.nc[2] + C.nc[2]) % C.nc[2];
                    const int wy = C.gbc[1] ? gy : (gy % C.nc[1] + C.nc[1]) % C.nc[1];
                    const int wx = C.gbc[0] ? gx : (gx % C.nc[0] + C.nc[0]) % C.nc[0];
                    const uint32_t gc = (uint32_t)(wx + C.nc[0] * (wy + C.nc[1] * wz));
                    for (uint32_t t = C.cell_start[gc]; t < C.cell_end[gc]; ++t) {
                        PsmCand pc;
                        psm_load_cand(C, t, pc);
                        if (pass == 1) { if (pc.id != id0 && pc.id != id1) psm_zero_dropped(P, C, r, pc); continue; }
                        double d[3]; int loc[3];
                        psm_rel(P, C, r, pc, d, loc);
                        if (!(cpl_dsc(pc.Rk, C.rc, cpl_dist(d)) > 0.0)) continue;
                        const uint32_t o0 = id0, o1 = id1;
                        dropped |= psm_select(pc.id, 0, id0, id1, c0, c1);
                        if (id0 != o0) { far1 = far0; far0 = pc; } else if (id1 != o1) far1 = pc;
                    }
                }
    }
    if (id0 == 0xffffffffu) { lb_collide_bgk(f, P.omega, rho, ux, uy, uz); return; }
    if (dropped) atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
    psm_cell(P, C, r, f, rho, ux, uy, uz, far0, far1, id1 == 0xffffffffu ? 1 : 2);
}

// One thread per cell, one block per 128-cell row segment.  The block first collects, together, the solids
// that can reach its row segment (walking the DEM grid cells around it) into shared memory; a row with no
// candidate runs the plain BGK path.
__global__ void __launch_bounds__(PSM_BLOCK, 4) lbm_psm_kernel(const double* __restrict__ fin, double* __restrict__ fout,
                                                               const __grid_constant__ LbmDev P,
                                                               const __grid_constant__ CplDev C)
{
    __shared__ PsmCand cand[PSM_MAXC];
    __shared__ int s_n;
    const int tid = threadIdx.x;
    const int x_first = blockIdx.x * PSM_BLOCK;
    const int x = x_first + tid, y = blockIdx.y, z = blockIdx.z;
    const bool active = x < P.nx;
    const long long cell = ((long long)z * P.ny + y) * P.nx + (active ? x : 0);
    double f[LEDDS_Q];
    if (active) {
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = __ldg(fin + (long long)q * P.N + cell);
    }
    if (tid == 0) s_n = 0;
    __syncthreads();
    {
        const int x_last = min(x_first + PSM_BLOCK - 1, P.nx - 1);
        const int rlo[3] = {x_first, y, z}, rhi[3] = {x_last, y, z};
        int clo[3], cnt[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int lo = (int)floor(rlo[a] * C.gs[a] + C.g0[a] - C.dg[a]);
            int hi = (int)floor(rhi[a] * C.gs[a] + C.g0[a] + C.dg[a]);
            if (C.gbc[a]) { lo = max(lo, 0); hi = min(hi, C.nc[a] - 1); }
            else if (hi - lo + 1 > C.nc[a]) hi = lo + C.nc[a] - 1;                    // whole periodic axis: once
            clo[a] = lo; cnt[a] = max(hi - lo + 1, 0);
        }
        const int total = cnt[0] * cnt[1] * cnt[2];
        for (int c = tid; c < total; c += PSM_BLOCK) {
            int g[3] = {clo[0] + c % cnt[0], clo[1] + (c / cnt[0]) % cnt[1], clo[2] + c / (cnt[0] * cnt[1])};
#pragma unroll
            for (int a = 0; a < 3; ++a)
                if (!C.gbc[a]) g[a] = (g[a] % C.nc[a] + C.nc[a]) % C.nc[a];
            const uint32_t gc = (uint32_t)(g[0] + C.nc[0] * (g[1] + C.nc[1] * g[2]));
            const uint32_t b = C.cell_start[gc], e = C.cell_end[gc];
            for (uint32_t t = b; t < e; ++t) {
                PsmCand pc;
                psm_load_cand(C, t, pc);
                // distance of the row (y, z fixed) from the sphere centre, nearest images
                const double dy = (double)(pc.fk[1] + cpl_offset(y, pc.fk[1], P.ny, !P.bc[1])) - pc.xk[1];
                const double dz = (double)(pc.fk[2] + cpl_offset(z, pc.fk[2], P.nz, !P.bc[2])) - pc.xk[2];
                const double reach = pc.Rk + C.rc;
                if (dy * dy + dz * dz > reach * reach * (1.0 + 1e-12)) continue;
                const int slot = atomicAdd(&s_n, 1);
                if (slot < PSM_MAXC) cand[slot] = pc;
            }
        }
    }
    __syncthreads();
    if (!active) return;
    const int ncand = s_n;
    const int r[3] = {x, y, z};
    double rho, ux, uy, uz;
    lb_moments(f, rho, ux, uy, uz);
    if (ncand == 0) {
        lb_collide_bgk(f, P.omega, rho, ux, uy, uz);
    } else if (ncand > PSM_MAXC) {
        // the out-of-line cold path gets a copy, so that f itself never has its address taken (it would
        // otherwise live in local memory for the whole kernel)
        double tmp[LEDDS_Q];
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) tmp[q] = f[q];
        psm_cell_global_search(P, C, r, tmp, rho, ux, uy, uz);
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = tmp[q];
    } else {
        uint32_t id0 = 0xffffffffu, id1 = 0xffffffffu;
        int c0 = 0, c1 = 0;
        bool dropped = false;
        for (int ci = 0; ci < ncand; ++ci) {
            const PsmCand& pc = cand[ci];
            double d[3]; int loc[3];
            psm_rel(P, C, r, pc, d, loc);
            if (!(cpl_dsc(pc.Rk, C.rc, cpl_dist(d)) > 0.0)) continue;
            dropped |= psm_select(pc.id, ci, id0, id1, c0, c1);
        }
        if (id0 == 0xffffffffu) {
            lb_collide_bgk(f, P.omega, rho, ux, uy, uz);
        } else {
            psm_cell(P, C, r, f, rho, ux, uy, uz, cand[c0], cand[c1], id1 == 0xffffffffu ? 1 : 2);
            if (dropped) {
                atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
                for (int ci = 0; ci < ncand; ++ci)
                    if (cand[ci].id != id0 && cand[ci].id != id1) psm_zero_dropped(P, C, r, cand[ci]);
            }
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
