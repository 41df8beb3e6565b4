// Fluid-solid coupling through partially saturated cells (PSM), Eq. (32)-(42),
// fused into the D3Q19 stream-collide pass, plus the coupled step driver.
//
//   cpl_raster_kernel  one warp per solid: marks the fluid cells the solid cuts (delta_sc > 0, Eq. 39-40) in the
//                      per-cell slot array, keeping the two lowest ids per cell (PAPER.md:515 n_s = 2) with
//                      two rounds of integer atomicMin.  Replaces the paper's per-cell neighbour search.
//   lbm_psm_kernel     one thread per cell: 19 coalesced loads + the cell's slot; empty slot -> plain BGK;
//                      else solid fraction Eq. (39)-(40), weights Eq. (36)-(37), PSM collision Eq. (32)-(35);
//                      streaming with boundaries; the (cell, solid) terms of Eq. (41)-(42) are summed over the
//                      block's row segment in shared memory in a fixed order and written as one row partial.
//   cpl_reduce_kernel  one warp per solid: fixed-order sum of its row partials -> F_sf, M_sf.  No floating
//                      point atomics and no sort over N_fluid (as PAPER.md:525-530 needs).
#include <math.h>

#include "psm_kernels.cuh"

// ------------------------------------------------------------------------------------ raster
// round 0: slots[cell].x = min id over the solids cutting the cell
// round 1: slots[cell].y = min id over the others; a third one raises LEDDS_ST_SOLID_OVERFLOW
__global__ void __launch_bounds__(128) cpl_raster_kernel(const LbmDev P, const CplDev C, int round)
{
    const int k = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (k >= C.n) return;
    const int nl[3] = {P.nx, P.ny, P.nz};
    double xk[3], Rk;
    int fk[3];
    cpl_solid(C, (uint32_t)k, xk, fk, Rk);
    const int S = C.S, S3 = S * S * S;
    bool overflow = false;
    for (int e = lane; e < S3; e += 32) {
        const int l[3] = {e % S, (e / S) % S, e / (S * S)};
        int rw[3];
        double d[3];
        bool inside = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int ri = fk[a] + (l[a] - C.H);
            d[a] = (double)ri - xk[a];
            if (P.bc[a]) { if (ri < 0 || ri >= nl[a]) inside = false; rw[a] = ri; }
            else rw[a] = ri - cpl_floordiv(ri, nl[a]) * nl[a];
        }
        if (!inside) continue;
        if (!(cpl_dsc(Rk, C.rc, cpl_dist(d)) > 0.0)) continue;
        uint2* slot = C.slots + (((long long)rw[2] * P.ny + rw[1]) * P.nx + rw[0]);
        if (round == 0) {
            atomicMin(&slot->x, (uint32_t)k);
        } else if (slot->x != (uint32_t)k) {
            if (atomicMin(&slot->y, (uint32_t)k) != PSM_EMPTY) overflow = true;
        }
    }
    if (overflow) atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
}

// ------------------------------------------------------------------------------------ collide + stream
__global__ void __launch_bounds__(PSM_BLOCK, 4) lbm_psm_kernel(const double* __restrict__ fin, double* __restrict__ fout,
                                                               const __grid_constant__ LbmDev P,
                                                               const __grid_constant__ CplDev C)
{
    __shared__ uint32_t sid[2][PSM_BLOCK];
    __shared__ double sval[6][2][PSM_BLOCK];
    const int tid = threadIdx.x;
    const int x = blockIdx.x * PSM_BLOCK + tid, y = blockIdx.y, z = blockIdx.z;
    const bool active = x < P.nx;
    uint32_t id[2] = {PSM_EMPTY, PSM_EMPTY};
    PsmRecord rec[2];
    if (active) {
        const long long cell = ((long long)z * P.ny + y) * P.nx + x;
        double f[LEDDS_Q];
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = __ldg(fin + (long long)q * P.N + cell);
        const uint2 slot = C.slots[cell];
        id[0] = slot.x; id[1] = slot.y;
        double rho, ux, uy, uz;
        lb_moments(f, rho, ux, uy, uz);
        if (id[0] == PSM_EMPTY) {
            lb_collide_bgk(f, P.omega, rho, ux, uy, uz);
        } else {
            C.slots[cell] = make_uint2(PSM_EMPTY, PSM_EMPTY);                         // consumed: free for the next step
            const int r[3] = {x, y, z};
            psm_cell(P, C, r, f, rho, ux, uy, uz, id, rec);
        }
        lb_push_store(fout, P, x, y, z, f, rho);
    }
    // ---- Eq. (41)-(42): fixed-order sum over the row segment of this block, one partial per (solid, row)
    if (!__syncthreads_or(id[0] != PSM_EMPTY)) return;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        sid[s][tid] = id[s];
        if (id[s] != PSM_EMPTY) {
#pragma unroll
            for (int c = 0; c < 6; ++c) sval[c][s][tid] = rec[s].v[c];
        }
    }
    __syncthreads();
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const uint32_t me = id[s];
        if (me == PSM_EMPTY) continue;
        // the first cell of this solid in the segment sums for all of them (they lie within S cells)
        bool head = true;
        for (int b = 1; b < C.S && b <= tid; ++b)
            if (sid[0][tid - b] == me || sid[1][tid - b] == me) { head = false; break; }
        if (!head) continue;
        double acc[6] = {rec[s].v[0], rec[s].v[1], rec[s].v[2], rec[s].v[3], rec[s].v[4], rec[s].v[5]};
        for (int b = 1; b < C.S && tid + b < PSM_BLOCK; ++b) {
            const int t = tid + b;
            const int s2 = sid[0][t] == me ? 0 : (sid[1][t] == me ? 1 : -1);
            if (s2 < 0) continue;
#pragma unroll
            for (int c = 0; c < 6; ++c) acc[c] += sval[c][s2][t];
        }
        const int seg = cpl_block_ordinal(rec[s].xu, P.nx, C.nbx) - cpl_block_ordinal(rec[s].x0, P.nx, C.nbx);
        const long long e = (long long)rec[s].row * C.nseg + seg;
        double* out = C.rows + e * 6;
#pragma unroll
        for (int c = 0; c < 6; ++c) out[c] = acc[c];
        C.stamps[e] = C.stamp;
    }
}

// ------------------------------------------------------------------------------------ reduce
// One warp per solid; lane -> entry map and the shuffle tree are fixed, so the sums are deterministic.
__global__ void __launch_bounds__(128) cpl_reduce_kernel(const CplDev C, double* __restrict__ f_hyd,
                                                         double* __restrict__ m_hyd)
{
    const int k = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (k >= C.n) return;
    const int E = C.S * C.S * C.nseg;
    const uint32_t* st = C.stamps + (long long)k * E;
    const double* rows = C.rows + (long long)k * E * 6;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int e = lane; e < E; e += 32) {
        if (st[e] != C.stamp) continue;
#pragma unroll
        for (int c = 0; c < 6; ++c) acc[c] += rows[(long long)e * 6 + c];
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        double v = acc[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        acc[c] = v;
    }
    if (lane == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            f_hyd[3 * k + c] = acc[c] * C.fscale;
            m_hyd[3 * k + c] = acc[3 + c] * C.mscale;
        }
    }
}

// ------------------------------------------------------------------------------------ host API
struct CplLayout { size_t slots, stamps, rows, total; };

static size_t cpl_align(size_t v) { return (v + 255) & ~(size_t)255; }

static int cpl_setup(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c, double r_max, CplDev* C,
                     CplLayout* L)
{
    if (!lbm || !dem || !c || c->n_sub < 1 || c->solid_fraction != 0 || !(c->dx > 0.0) || !(c->rho_f > 0.0) || !(r_max > 0.0))
        return LEDDS_EINVAL;
    const double rc = cbrt(3.0 / (4.0 * 3.14159265358979323846));           // Eq. (40), dx = 1
    const double Dt = c->n_sub * dem->d.dt;
    C->n = dem->d.n;
    C->rc = rc;
    C->inv_dx = 1.0 / c->dx;
    C->vscale = Dt / c->dx;
    C->wscale = Dt;
    C->fscale = c->rho_f * pow(c->dx, 4) / (Dt * Dt);
    C->mscale = c->rho_f * pow(c->dx, 5) / (Dt * Dt);
    const int nl[3] = {lbm->d.nx, lbm->d.ny, lbm->d.nz};
    C->H = (int)ceil(r_max / c->dx + rc);
    C->S = 2 * C->H + 2;
    if (C->S > PSM_BLOCK) return LEDDS_EINVAL;                              // a row of the box spans <= 2 blocks (+ seam)
    C->nbx = (nl[0] + PSM_BLOCK - 1) / PSM_BLOCK;
    C->nseg = (lbm->d.bc[0] || nl[0] % PSM_BLOCK == 0) ? 2 : 3;
    for (int a = 0; a < 3; ++a) {
        C->origin[a] = c->origin[a];
        if (dem->d.bc[a] != lbm->d.bc[a]) return LEDDS_EINVAL;              // same topology on both grids
        if (!lbm->d.bc[a] && nl[a] < 2 * C->S) return LEDDS_EINVAL;         // unambiguous nearest image (G33)
    }
    const size_t N = (size_t)lbm->d.N, E = (size_t)C->n * C->S * C->S * C->nseg;
    if ((double)C->n * C->S * C->S > 2.0e9) return LEDDS_EINVAL;
    L->slots = 0;
    L->stamps = cpl_align(N * sizeof(uint2));
    L->rows = L->stamps + cpl_align(E * sizeof(uint32_t));
    L->total = L->rows + cpl_align(E * 6 * sizeof(double));
    return LEDDS_OK;
}

extern "C" int ledds_cpl_workspace_bytes(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c,
                                         const double r_max, size_t* bytes)
{
    CplDev C;
    CplLayout L;
    const int rc = cpl_setup(lbm, dem, c, r_max, &C, &L);
    if (rc) return rc;
    if (!bytes) return LEDDS_EINVAL;
    *bytes = L.total;
    return LEDDS_OK;
}

extern "C" int ledds_cpl_init(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c, double r_max,
                              void* cpl_scratch, void* stream)
{
    CplDev C;
    CplLayout L;
    const int rc = cpl_setup(lbm, dem, c, r_max, &C, &L);
    if (rc) return rc;
    if (!cpl_scratch) return LEDDS_EINVAL;
    if (!ledds_aligned16(cpl_scratch)) return LEDDS_EALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    char* base = static_cast<char*>(cpl_scratch);
    if (cudaMemsetAsync(base + L.slots, 0xff, L.stamps - L.slots, st) != cudaSuccess ||     // all slots PSM_EMPTY
        cudaMemsetAsync(base + L.stamps, 0, L.rows - L.stamps, st) != cudaSuccess)          // no partial is current
        return LEDDS_ECUDA;
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
    CplLayout L;
    int rc = cpl_setup(lbm, dem, c, r_max, &C, &L);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const DemScratch& s = dem->s;
    char* sc = static_cast<char*>(scratch);
    char* cs = static_cast<char*>(cpl_scratch);
    C.x = x;
    C.vp = reinterpret_cast<const double*>(sc + s.vp);
    C.wp = reinterpret_cast<const double*>(sc + s.wp);
    C.radius = radius;
    C.slots = reinterpret_cast<uint2*>(cs + L.slots);
    C.stamps = reinterpret_cast<uint32_t*>(cs + L.stamps);
    C.rows = reinterpret_cast<double*>(cs + L.rows);
    C.status = status;
    const LbmDev& d = lbm->d;
    const size_t half = (size_t)LEDDS_Q * d.N;
    if (d.ny > 65535 || d.nz > 65535) return LEDDS_EINVAL;
    const unsigned warp_blocks = (unsigned)(((long long)C.n * 32 + 127) / 128);
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
        C.stamp = (uint32_t)(lbm->steps % 0xfffffffell) + 1u;
        ledds_prof_start(LEDDS_K_CPL_RASTER, st);
        cpl_raster_kernel<<<warp_blocks, 128, 0, st>>>(d, C, 0);
        cpl_raster_kernel<<<warp_blocks, 128, 0, st>>>(d, C, 1);
        ledds_prof_stop(LEDDS_K_CPL_RASTER, st);
        ledds_count_launch(1);
        LEDDS_CHECK_LAUNCH();
        dim3 block(PSM_BLOCK), grid(C.nbx, d.ny, d.nz);
        ledds_prof_start(LEDDS_K_LBM, st);
        lbm_psm_kernel<<<grid, block, 0, st>>>(f + lbm->parity * half, f + (1 - lbm->parity) * half, d, C);
        ledds_prof_stop(LEDDS_K_LBM, st);
        LEDDS_CHECK_LAUNCH();
        lbm->parity ^= 1;
        lbm->steps++;
        ledds_prof_start(LEDDS_K_CPL_REDUCE, st);
        cpl_reduce_kernel<<<warp_blocks, 128, 0, st>>>(C, f_hyd, m_hyd);
        ledds_prof_stop(LEDDS_K_CPL_REDUCE, st);
        LEDDS_CHECK_LAUNCH();
        rc = ledds_dem_kick(dem, v, w, a, alpha, radius, f_hyd, m_hyd, scratch, status, st);
        if (rc) return rc;
        dem->steps++;
    }
    return LEDDS_OK;
}
