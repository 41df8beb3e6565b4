// Fluid-solid coupling through partially saturated cells (PSM), Eq. (32)-(42),
// fused into the D3Q19 stream-collide pass, plus the coupled step driver.
//
//   cpl_raster_kernel  one warp per solid: converts the solid's state to lattice units and marks the fluid
//                      cells it cuts (delta_sc > 0, Eq. 39-40) in the per-cell slot array, keeping the two lowest
//                      ids per cell (PAPER.md:515 n_s = 2) with two rounds of integer atomicMin.  Replaces the
//                      paper's per-cell neighbour search.
//   lbm_psm_kernel     one thread per cell: 19 coalesced loads + the cell's slot.  A warp without a solid runs
//                      the plain BGK path; otherwise all its lanes run the PSM collision Eq. (32)-(37) (B = 0
//                      where there is no solid), stream with boundaries, and the (cell, solid) terms of
//                      Eq. (41)-(42) are summed over runs of consecutive lanes by warp shuffles in a fixed
//                      order; the first lane of a run stores one partial.
//   cpl_reduce_kernel  one warp per solid: fixed-order sum of its partials -> F_sf, M_sf.  No floating point
//                      atomics and no sort over N_fluid (as PAPER.md:525-530 needs).
#include <math.h>

#include "psm_kernels.cuh"

// ------------------------------------------------------------------------------------ raster
// slots[cell] = the two lowest ids of the solids cutting the cell (x < y), kept with a 64-bit compare-and-swap;
// a third solid raises LEDDS_ST_SOLID_OVERFLOW.  Also writes sol[k].  A warp walks the rows of the solid's
// box, 32 / Spad rows at a time (Spad = S rounded up to a power of two), one lane per cell.
__global__ void __launch_bounds__(128) cpl_raster_kernel(const LbmDev P, const CplDev C, int spad_log2)
{
    const int k = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (k >= C.n) return;
    double xk[3];
    int fk[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        xk[a] = (C.x[3 * k + a] - C.origin[a]) * C.inv_dx;
        fk[a] = (int)floor(xk[a]);
    }
    const double Rk = C.radius[k] * C.inv_dx;
    if (lane < 10) {
        double v;
        if (lane < 3) v = xk[lane];
        else if (lane == 3) v = Rk;
        else if (lane < 7) v = C.vp[3 * k + lane - 4] * C.vscale;
        else v = C.wp[3 * k + lane - 7] * C.wscale;
        C.sol[(size_t)k * 10 + lane] = v;
    }
    const int S = C.S;
    const int sub = lane >> spad_log2, lx0 = lane & ((1 << spad_log2) - 1), rows_per_iter = 32 >> spad_log2;
    const int xstep = 1 << spad_log2;
    bool overflow = false;
    for (int lz = 0; lz < S; ++lz) {
        int rz = fk[2] + lz - C.H;
        const double dz = (double)rz - xk[2];
        if (P.bc[2]) { if (rz < 0 || rz >= P.nz) continue; }
        else rz = rz < 0 ? rz + P.nz : (rz >= P.nz ? rz - P.nz : rz);
        for (int ly0 = 0; ly0 < S; ly0 += rows_per_iter) {
            const int ly = ly0 + sub;
            int ry = fk[1] + ly - C.H;
            const double dy = (double)ry - xk[1];
            bool row_ok = ly < S;
            if (P.bc[1]) { if (ry < 0 || ry >= P.ny) row_ok = false; }
            else ry = ry < 0 ? ry + P.ny : (ry >= P.ny ? ry - P.ny : ry);
            for (int lx = lx0; lx < S; lx += xstep) {
                int rx = fk[0] + lx - C.H;
                const double d[3] = {(double)rx - xk[0], dy, dz};
                if (P.bc[0]) { if (rx < 0 || rx >= P.nx) continue; }
                else rx = rx < 0 ? rx + P.nx : (rx >= P.nx ? rx - P.nx : rx);
                if (!row_ok || !cpl_cuts(Rk, C.rc, d)) continue;
                unsigned long long* slot = reinterpret_cast<unsigned long long*>(C.slots + (((long long)rz * P.ny + ry) * P.nx + rx));
                unsigned long long old = *slot;
                for (;;) {
                    const uint32_t a = (uint32_t)old, b = (uint32_t)(old >> 32);   // uint2 {x = low word, y = high word}, a <= b
                    if ((uint32_t)k > b) { overflow = true; break; }                // two lower ids are already there
                    const uint32_t na = (uint32_t)k < a ? (uint32_t)k : a, nb = (uint32_t)k < a ? a : (uint32_t)k;
                    const unsigned long long seen = atomicCAS(slot, old, ((unsigned long long)nb << 32) | na);
                    if (seen == old) { overflow = overflow || b != PSM_EMPTY; break; }   // b was pushed out
                    old = seen;
                }
            }
        }
    }
    if (overflow) atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
}

// ------------------------------------------------------------------------------------ collide + stream
__global__ void __launch_bounds__(PSM_BLOCK, 4) lbm_psm_kernel(const double* __restrict__ fin, double* __restrict__ fout,
                                                               const __grid_constant__ LbmDev P,
                                                               const __grid_constant__ CplDev C)
{
    const int x = blockIdx.x * PSM_BLOCK + threadIdx.x, y = blockIdx.y, z = blockIdx.z;
    const bool active = x < P.nx;
    const long long cell = ((long long)z * P.ny + y) * P.nx + (active ? x : 0);
    uint32_t id[2] = {PSM_EMPTY, PSM_EMPTY};
    double f[LEDDS_Q];
    if (active) {
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = __ldg(fin + (long long)q * P.N + cell);
        const uint2 slot = C.slots[cell];
        id[0] = slot.x; id[1] = slot.y;
    } else {
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = lb_w(q);
    }
    double rho, ux, uy, uz;
    lb_moments(f, rho, ux, uy, uz);
    const bool any1 = __any_sync(0xffffffffu, id[0] != PSM_EMPTY);
    const bool any2 = __any_sync(0xffffffffu, id[1] != PSM_EMPTY);
    double rec[2][6];
    int ent[2];
    if (!any1) {
        lb_collide_bgk(f, P.omega, rho, ux, uy, uz);
    } else {
        if (id[0] != PSM_EMPTY) C.slots[cell] = make_uint2(PSM_EMPTY, PSM_EMPTY);     // consumed: free for the next step
        if (!any2) psm_cell<1>(P, C, x, y, z, f, rho, ux, uy, uz, id, rec, ent);
        else psm_cell<2>(P, C, x, y, z, f, rho, ux, uy, uz, id, rec, ent);
    }
    if (active) lb_push_store(fout, P, x, y, z, f, rho);
    if (any1) psm_run_reduce(C, id[0], ent[0], rec[0]);
    if (any2) psm_run_reduce(C, id[1], ent[1], rec[1]);
}

// ------------------------------------------------------------------------------------ reduce
// One warp per solid; lane -> entry map and the shuffle tree are fixed, so the sums are deterministic.
__global__ void __launch_bounds__(128) cpl_reduce_kernel(const CplDev C, double* __restrict__ f_hyd,
                                                         double* __restrict__ m_hyd)
{
    const int k = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (k >= C.n) return;
    const int S3 = C.S * C.S * C.S;                                                  // multiple of 8
    uint32_t* fl = reinterpret_cast<uint32_t*>(C.flags + (size_t)k * S3);
    const double* box = C.box + (size_t)k * S3 * 6;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int w4 = lane; w4 < S3 / 4; w4 += 32) {
        uint32_t m = fl[w4];
        if (!m) continue;
        fl[w4] = 0u;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            if (!((m >> (8 * b)) & 0xffu)) continue;
            const double2* in = reinterpret_cast<const double2*>(box + (size_t)(4 * w4 + b) * 6);
            const double2 a0 = in[0], a1 = in[1], a2 = in[2];
            acc[0] += a0.x; acc[1] += a0.y; acc[2] += a1.x; acc[3] += a1.y; acc[4] += a2.x; acc[5] += a2.y;
        }
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
struct CplLayout { size_t slots, sol, flags, box, total; };

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
    C->inv_2rc = 1.0 / (2.0 * rc);
    C->inv_dx = 1.0 / c->dx;
    C->vscale = Dt / c->dx;
    C->wscale = Dt;
    C->fscale = c->rho_f * pow(c->dx, 4) / (Dt * Dt);
    C->mscale = c->rho_f * pow(c->dx, 5) / (Dt * Dt);
    const int nl[3] = {lbm->d.nx, lbm->d.ny, lbm->d.nz};
    C->H = (int)ceil(r_max / c->dx + rc);
    C->S = 2 * C->H + 2;
    if (C->S > 256) return LEDDS_EINVAL;
    for (int a = 0; a < 3; ++a) {
        C->origin[a] = c->origin[a];
        if (dem->d.bc[a] != lbm->d.bc[a]) return LEDDS_EINVAL;              // same topology on both grids
        if (!lbm->d.bc[a] && nl[a] < 2 * C->S) return LEDDS_EINVAL;         // unambiguous nearest image (G33)
    }
    const size_t N = (size_t)lbm->d.N, S3 = (size_t)C->S * C->S * C->S, E = (size_t)C->n * S3;   // S even: S3 % 8 == 0
    L->slots = 0;
    L->sol = cpl_align(N * sizeof(uint2));
    L->flags = L->sol + cpl_align((size_t)C->n * 10 * sizeof(double));
    L->box = L->flags + cpl_align(E);
    L->total = L->box + cpl_align(E * 6 * sizeof(double));
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
    if (cudaMemsetAsync(base + L.slots, 0xff, L.sol - L.slots, st) != cudaSuccess ||        // all slots PSM_EMPTY
        cudaMemsetAsync(base + L.flags, 0, L.box - L.flags, st) != cudaSuccess)             // no partial pending
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
    C.sol = reinterpret_cast<double*>(cs + L.sol);
    C.flags = reinterpret_cast<uint8_t*>(cs + L.flags);
    C.box = reinterpret_cast<double*>(cs + L.box);
    C.status = status;
    const LbmDev& d = lbm->d;
    const size_t half = (size_t)LEDDS_Q * d.N;
    if (d.ny > 65535 || d.nz > 65535) return LEDDS_EINVAL;
    int spad_log2 = 0;
    while ((1 << spad_log2) < C.S && spad_log2 < 5) ++spad_log2;
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
        ledds_prof_start(LEDDS_K_CPL_RASTER, st);
        cpl_raster_kernel<<<warp_blocks, 128, 0, st>>>(d, C, spad_log2);
        ledds_prof_stop(LEDDS_K_CPL_RASTER, st);
        LEDDS_CHECK_LAUNCH();
        dim3 block(PSM_BLOCK), grid((d.nx + PSM_BLOCK - 1) / PSM_BLOCK, d.ny, d.nz);
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
