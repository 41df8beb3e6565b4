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
// a third solid raises LEDDS_ST_SOLID_OVERFLOW; a cell that gets its second solid is appended to list2.
// Also writes sol[k].  A warp walks the rows of the solid's box, 32 / Spad rows at a time (Spad = S rounded
// up to a power of two), one lane per cell.  RASTER_BATCH optimistic swaps (expecting an empty slot) are in
// flight before the first answer is looked at, so the walk is not a chain of memory round trips.
#define RASTER_BATCH 6
#define PSM_EMPTY64 0xffffffffffffffffull

// returns true when this insert gave the cell its second solid
__device__ __forceinline__ bool raster_insert(unsigned long long* slot, unsigned long long old, uint32_t k, bool& overflow)
{
    for (;;) {
        const uint32_t a = (uint32_t)old, b = (uint32_t)(old >> 32);           // uint2 {x = low word, y = high word}, a <= b
        if (k > b) { overflow = true; return false; }                           // two lower ids are already there
        const uint32_t na = k < a ? k : a, nb = k < a ? a : k;
        const unsigned long long seen = atomicCAS(slot, old, ((unsigned long long)nb << 32) | na);
        if (seen == old) {
            if (b != PSM_EMPTY) { overflow = true; return false; }              // b was pushed out
            return a != PSM_EMPTY;
        }
        old = seen;
    }
}

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
    const int iters_y = (S + rows_per_iter - 1) / rows_per_iter, iters = S * iters_y;
    bool overflow = false;
    for (int lxb = 0; lxb < S; lxb += xstep) {                                  // one trip unless S > 32; uniform
        const int lx = lxb + lx0;
        int rx = fk[0] + lx - C.H;
        const double dx = (double)rx - xk[0];
        bool xok = lx < S;
        if (P.bc[0]) xok = xok && rx >= 0 && rx < P.nx;
        else rx = rx < 0 ? rx + P.nx : (rx >= P.nx ? rx - P.nx : rx);
        for (int it0 = 0; it0 < iters; it0 += RASTER_BATCH) {
            unsigned long long* slot[RASTER_BATCH];
            unsigned long long seen[RASTER_BATCH];
            uint32_t cell[RASTER_BATCH];
#pragma unroll
            for (int b = 0; b < RASTER_BATCH; ++b) {
                const int it = it0 + b;
                const int lz = it / iters_y, ly = (it - lz * iters_y) * rows_per_iter + sub;
                int rz = fk[2] + lz - C.H, ry = fk[1] + ly - C.H;
                const double d[3] = {dx, (double)ry - xk[1], (double)rz - xk[2]};
                bool ok = xok && it < iters && ly < S;
                if (P.bc[2]) ok = ok && rz >= 0 && rz < P.nz;
                else rz = rz < 0 ? rz + P.nz : (rz >= P.nz ? rz - P.nz : rz);
                if (P.bc[1]) ok = ok && ry >= 0 && ry < P.ny;
                else ry = ry < 0 ? ry + P.ny : (ry >= P.ny ? ry - P.ny : ry);
                ok = ok && cpl_cuts(Rk, C.rc, d);
                slot[b] = nullptr;
                seen[b] = PSM_EMPTY64;
                cell[b] = 0u;
                if (ok) {
                    cell[b] = (uint32_t)(((long long)rz * P.ny + ry) * P.nx + rx);
                    slot[b] = reinterpret_cast<unsigned long long*>(C.slots + cell[b]);
                    seen[b] = atomicCAS(slot[b], PSM_EMPTY64, ((unsigned long long)PSM_EMPTY << 32) | (uint32_t)k);
                }
            }
#pragma unroll
            for (int b = 0; b < RASTER_BATCH; ++b) {
                bool second = false;
                if (slot[b] && seen[b] != PSM_EMPTY64) second = raster_insert(slot[b], seen[b], (uint32_t)k, overflow);
                // one list2 append per warp, in lane (= x) order so that neighbouring cells stay neighbours
                const unsigned m = __ballot_sync(0xffffffffu, second);
                if (m) {
                    uint32_t base = 0;
                    if (lane == __ffs(m) - 1) base = atomicAdd(C.list2, (uint32_t)__popc(m));
                    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
                    const uint32_t at = base + (uint32_t)__popc(m & ((1u << lane) - 1u));
                    if (second && at < C.list2_cap) C.list2[1 + at] = cell[b];
                }
            }
        }
    }
    if (overflow) atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
}

// ------------------------------------------------------------------------------------ collide + stream
// Cells cut by two solids are left to lbm_psm2_kernel: here they take the plain collision (overwritten later)
// and contribute no partial.
__global__ void __launch_bounds__(PSM_BLOCK, 5) lbm_psm_kernel(const double* __restrict__ fin, double* __restrict__ fout,
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
        if (slot.y == PSM_EMPTY) id[0] = slot.x;
    } else {
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = lb_w(q);
    }
    double rho, ux, uy, uz;
    lb_moments(f, rho, ux, uy, uz);
    const bool any1 = __any_sync(0xffffffffu, id[0] != PSM_EMPTY);
    double rec[2][6];
    int ent[2];
    if (!any1) {
        lb_collide_bgk(f, P.omega, rho, ux, uy, uz);
    } else {
        if (id[0] != PSM_EMPTY) C.slots[cell] = make_uint2(PSM_EMPTY, PSM_EMPTY);     // consumed: free for the next step
        psm_cell<1>(P, C, x, y, z, f, rho, ux, uy, uz, id, rec, ent);
    }
    if (active) lb_push_store(fout, P, x, y, z, f, rho);
    if (any1) psm_run_reduce(C, id[0], ent[0], rec[0]);
}

// The cells cut by two solids (list2), one thread each: same step as above with both solids; every cell stores
// its own two partials.  Runs after lbm_psm_kernel on the same stream and overwrites what that wrote for them.
__global__ void __launch_bounds__(128) lbm_psm2_kernel(const double* __restrict__ fin, double* __restrict__ fout,
                                                       const __grid_constant__ LbmDev P,
                                                       const __grid_constant__ CplDev C)
{
    const uint32_t count = min(C.list2[0], C.list2_cap);
    const uint32_t padded = (count + 31u) & ~31u;                                    // whole warps stay together
    for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < padded; t += gridDim.x * blockDim.x) {
        const bool on = t < count;
        const uint32_t cell = on ? C.list2[1 + t] : 0u;
        const int x = (int)(cell % (uint32_t)P.nx), y = (int)((cell / (uint32_t)P.nx) % (uint32_t)P.ny);
        const int z = (int)(cell / ((uint32_t)P.nx * (uint32_t)P.ny));
        double f[LEDDS_Q];
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = __ldg(fin + (long long)q * P.N + cell);
        uint32_t id[2] = {PSM_EMPTY, PSM_EMPTY};
        if (on) {
            const uint2 slot = C.slots[cell];
            C.slots[cell] = make_uint2(PSM_EMPTY, PSM_EMPTY);
            id[0] = slot.x; id[1] = slot.y;
        }
        double rho, ux, uy, uz;
        lb_moments(f, rho, ux, uy, uz);
        double rec[2][6];
        int ent[2];
        psm_cell<2>(P, C, x, y, z, f, rho, ux, uy, uz, id, rec, ent);
        if (on) lb_push_store(fout, P, x, y, z, f, rho);
        // neighbours in the list are mostly neighbours on the lattice cut by the same two solids
        psm_run_reduce(C, id[0], ent[0], rec[0]);
        psm_run_reduce(C, id[1], ent[1], rec[1]);
    }
}

// ------------------------------------------------------------------------------------ reduce
// One warp per solid; lane -> entry map and the shuffle tree are fixed, so the sums are deterministic.
// Each lane takes 16 flags at a time (one 16-byte load) and reads the flagged partials.
__global__ void __launch_bounds__(128) cpl_reduce_kernel(const CplDev C, double* __restrict__ f_hyd,
                                                         double* __restrict__ m_hyd)
{
    const int k = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (blockIdx.x == 0 && threadIdx.x == 0) C.list2[0] = 0u;                        // list worked through: empty it
    if (k >= C.n) return;
    const int S3 = C.S * C.S * C.S;                                                  // multiple of 8
    uint2* fl = reinterpret_cast<uint2*>(C.flags + (size_t)k * S3);
    const double2* box = reinterpret_cast<const double2*>(C.box + (size_t)k * S3 * 6);
    double acc[6] = {0, 0, 0, 0, 0, 0};
    const double2 zero = make_double2(0.0, 0.0);
    for (int w8 = lane; w8 < S3 / 8; w8 += 32) {
        const uint2 m = fl[w8];
        if (!(m.x | m.y)) continue;
        fl[w8] = make_uint2(0u, 0u);
        double2 a[8][3];
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            const bool on = (((b < 4 ? m.x : m.y) >> (8 * (b & 3))) & 0xffu) != 0u;
            const double2* in = box + (size_t)(8 * w8 + b) * 3;
            a[b][0] = on ? in[0] : zero; a[b][1] = on ? in[1] : zero; a[b][2] = on ? in[2] : zero;
        }
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            acc[0] += a[b][0].x; acc[1] += a[b][0].y; acc[2] += a[b][1].x;
            acc[3] += a[b][1].y; acc[4] += a[b][2].x; acc[5] += a[b][2].y;
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
struct CplLayout { size_t slots, sol, list2, flags, box, total; uint32_t list2_cap; };

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
    L->list2 = L->sol + cpl_align((size_t)C->n * 10 * sizeof(double));
    L->list2_cap = (uint32_t)(E < N ? E : N);                              // every 2-solid cell lies in some solid's box
    L->flags = L->list2 + cpl_align(((size_t)L->list2_cap + 1) * sizeof(uint32_t));
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
        cudaMemsetAsync(base + L.list2, 0, 256, st) != cudaSuccess ||                       // list2 count
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
    C.list2 = reinterpret_cast<uint32_t*>(cs + L.list2);
    C.list2_cap = L.list2_cap;
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
        ledds_prof_start(LEDDS_K_CPL_PSM2, st);
        lbm_psm2_kernel<<<148 * 4, 128, 0, st>>>(f + lbm->parity * half, f + (1 - lbm->parity) * half, d, C);
        ledds_prof_stop(LEDDS_K_CPL_PSM2, st);
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
