// Fluid-solid coupling through partially saturated cells (PSM), Eq. (32)-(42),
// fused into the D3Q19 stream-collide pass, plus the coupled step driver.
//
//   cpl_raster_kernel  one thread per (solid, row of its bounding box): finds the run of fluid cells the solid
//                      cuts in that row (delta_sc > 0, Eq. 39-40) and enters the solid in their slots, keeping
//                      the two lowest ids per cell (PAPER.md:515 n_s = 2) with a 64-bit compare-and-swap.
//                      Replaces the paper's per-cell neighbour search.
//   lbm_psm_kernel     one thread per cell: 19 coalesced loads + the cell's slot.  A warp without a solid runs
//                      the plain BGK path; otherwise all its lanes run the PSM collision Eq. (32)-(37) (B = 0
//                      where there is no solid; the rarer second solid of a cell is parked in shared memory),
//                      stream with boundaries, and the (cell, solid) terms of Eq. (41)-(42) are summed over
//                      runs of consecutive lanes by warp shuffles; the first lane of a run adds the sum to the
//                      solid's 2^-83 fixed-point accumulators with integer reductions.
//   cpl_finish_kernel  fixed point -> F_sf, M_sf.  No floating point atomics and no sort over N_fluid (as
//                      PAPER.md:525-530 needs); the integer sums are exact and order-independent.
#include <math.h>

#include "psm_kernels.cuh"

// ------------------------------------------------------------------------------------ raster

#define RASTER_BATCH 6

// sol[k] = the solid in lattice units (one thread per home slot of the DEM state; k = the particle's id)
__global__ void cpl_solid_kernel(const CplDev C)
{
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= C.n) return;
    const double4 r = C.hx[h];
    const double xr[3] = {r.x, r.y, r.z};
    const double* pv = C.pvw + 6 * (size_t)h;
    double* o = C.sol + (size_t)C.hid[h] * 10;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        o[a] = (xr[a] - C.origin[a]) / C.dx;                     // divisions, as PAPER.md:256 states the conversion
        o[4 + a] = pv[a] * C.vscale;
        o[7 + a] = pv[3 + a] * C.wscale;
    }
    o[3] = r.w / C.dx;
    if (r.w > C.r_max) atomicOr(C.status, LEDDS_ST_RADIUS_RANGE);   // its box (H from r_max) would truncate it
}

// Eq. (38) in two kernels: every (solid, cell of its bounding box) is classified -- by the distance of its centre where
// that settles it, else from its nearest and farthest sample point (all inside: 1, all outside: 0); the cells the
// surface crosses go to a list, and the second kernel counts their 10^3 points with one thread per listed cell, so
// that its warps hold only cells that need it.
__device__ __forceinline__ void cpl_box_cell(const CplDev& C, long long t, double* d, double& Rk)
{
    const int S = C.S, S3 = S * S * S;
    const int k = (int)(t / S3);
    const int e = (int)(t - (long long)k * S3), lz = e / (S * S), ly = (e / S) % S, lx = e % S;
    const double* o = C.sol + (size_t)k * 10;
    d[0] = (double)((int)floor(o[0]) + lx - C.H) - o[0];
    d[1] = (double)((int)floor(o[1]) + ly - C.H) - o[1];
    d[2] = (double)((int)floor(o[2]) + lz - C.H) - o[2];
    Rk = o[3];
}

// one thread per (solid, row of its box): the row's cells one after the other (the index arithmetic, the solid's record
// and the y, z parts of the distances once per row)
__global__ void __launch_bounds__(256) cpl_beta_classify_kernel(const CplDev C)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int S = C.S, S2 = S * S;
    const bool in = t < (long long)C.n * S2;
    const int k = in ? (int)(t / S2) : 0;
    const int r = (int)(t - (long long)k * S2), lz = r / S, ly = r - lz * S;
    const double* o = C.sol + (size_t)k * 10;
    const double Rk = o[3], ro = Rk + 0.78, ri = Rk - 0.78;
    const int fx = (int)floor(o[0]);
    const double dy = (double)((int)floor(o[1]) + ly - C.H) - o[1], dz = (double)((int)floor(o[2]) + lz - C.H) - o[2];
    const double dyz2 = dy * dy + dz * dz;
    const int lane = threadIdx.x & 31;
    // First the whole row by the distance of the cell centres: every sample point lies within 0.45 sqrt(3) = 0.7795 of
    // its cell's centre, so a centre further than R + 0.78 from the solid's (nearer than R - 0.78) has all its points
    // outside (inside) whatever the rounding of the point tests (the slack, 6e-4, is twelve orders above it).  The cells
    // of the shell in between -- two to four of a row -- are remembered in a bit mask and looked at point by point in a
    // second loop, which runs as often as the lane with the most shell cells needs, not once per cell of the row.
    for (int lx0 = 0; lx0 < S; lx0 += 64) {                                        // 64 cells of the row at a time (one mask)
    unsigned long long shell = 0ull;
    for (int lx = lx0; lx < min(S, lx0 + 64); ++lx) {
        if (!in) break;
        const double dx = (double)(fx + lx - C.H) - o[0];
        const double d2 = dx * dx + dyz2;
        if (d2 > ro * ro) C.betabox[t * S + lx] = 0.0;
        else if (ri > 0.0 && d2 < ri * ri) C.betabox[t * S + lx] = 1.0;
        else shell |= 1ull << (lx - lx0);
    }
    while (__any_sync(0xffffffffu, shell != 0ull)) {
        const bool has = shell != 0ull;
        const int lx = lx0 + (has ? __ffsll((long long)shell) - 1 : 0);
        shell &= shell - 1ull;
        const long long cell = t * S + lx;                                         // = (k S^2 + r) S + lx
        double beta = 0.0;
        if (has) {
            const double d[3] = {(double)(fx + lx - C.H) - o[0], dy, dz};
            SubdivPoints p;
            cpl_subdiv_points(d, Rk, p);
            beta = cpl_beta_classify(p);
            C.betabox[cell] = beta;
        }
        const bool todo = has && beta < 0.0;
        const unsigned m = __ballot_sync(0xffffffffu, todo);                        // one list append per warp
        if (m) {
            const int leader = __ffs(m) - 1;
            uint32_t base = 0;
            if (lane == leader) base = atomicAdd(C.blist, (uint32_t)__popc(m));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (todo) C.blist[1 + base + __popc(m & ((1u << lane) - 1u))] = (uint32_t)cell;
        }
    }
    }
}

__global__ void __launch_bounds__(256, 3) cpl_beta_count_kernel(const CplDev C)
{
    __shared__ double zs[PSM_NSUB][256];
    const uint32_t count = C.blist[0];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < count; i += gridDim.x * blockDim.x) {
        const long long t = C.blist[1 + i];
        double d[3], Rk;
        cpl_box_cell(C, t, d, Rk);
        SubdivPoints p;
        cpl_subdiv_points(d, Rk, p);
        C.betabox[t] = cpl_beta_count(p, &zs[0][threadIdx.x], 256);
    }
}

// thread t -> solid k = t / S^2, row (ly, lz) = t % S^2 of its box.
// Every cut cell gets slots[cell].x = min(x, k).  The value that was there tells who lost the cell: the
// newcomer if a lower id was already in, else the id it displaced; the loser is entered into slots[cell].y
// the same way.  Every solid but the lowest is a loser exactly once, so y ends as the second lowest id
// whatever the order of arrival (the two lowest ids), and a second loser is a third solid
// (LEDDS_ST_SOLID_OVERFLOW).  Only cells shared by two solids pay the second atomic.
template <bool SUBDIV>
__global__ void __launch_bounds__(256) cpl_raster_kernel(const LbmDev P, const CplDev C)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int S = C.S, S2 = S * S;
    const int k = (int)(t / S2);
    if (k >= C.n) return;
    const int r = (int)(t - (long long)k * S2), lz = r / S, ly = r - lz * S;
    const double* o = C.sol + (size_t)k * 10;
    const double xk[3] = {o[0], o[1], o[2]}, Rk = o[3];
    const int fk[3] = {(int)floor(xk[0]), (int)floor(xk[1]), (int)floor(xk[2])};
    int ry = fk[1] + ly - C.H, rz = fk[2] + lz - C.H;
    double d[3] = {0.0, (double)ry - xk[1], (double)rz - xk[2]};
    if (P.bc[1]) { if (ry < 0 || ry >= P.ny) return; }
    else ry = ry < 0 ? ry + P.ny : (ry >= P.ny ? ry - P.ny : ry);
    if (P.bc[2]) { if (rz < 0 || rz >= P.nz) return; }
    else rz = rz < 0 ? rz + P.nz : (rz >= P.nz ? rz - P.nz : rz);
    const int lo = fk[0] - C.H, hi = fk[0] + C.H + 1;                          // the box
    int xa, xb;
    auto cuts = [&](int xi) { d[0] = (double)xi - xk[0]; return cpl_cuts(Rk, C.rc, d); };
    if (SUBDIV) {
        // Eq. (38): beta of every cell of the row, kept in the solid's box; the cut cells (beta > 0) are a run
        const double* brow = C.betabox + ((size_t)k * S2 + r) * S;
        xa = hi + 1; xb = lo - 1;
        for (int xi = lo; xi <= hi; ++xi)                                       // written by cpl_beta_kernel
            if (brow[xi - lo] > 0.0) { xa = min(xa, xi); xb = max(xb, xi); }
        if (xa > xb) return;
    } else {
        // the cut cells of the row are the run [xa, xb] around x_k (the squared distance grows with |dx| also in
        // floating point): estimate its ends, then settle them with the exact test
        const double s = Rk + C.rc, h2 = s * s - (d[1] * d[1] + d[2] * d[2]);
        if (h2 < -1e-9 * s * s) return;
        const double w = sqrt(h2 > 0.0 ? h2 : 0.0);
        xa = max(lo, (int)ceil(xk[0] - w)); xb = min(hi, (int)floor(xk[0] + w));
        if (xa > xb) { xa = xb = min(hi, max(lo, (int)floor(xk[0] + 0.5))); if (!cuts(xa)) return; }
        while (xa <= xb && !cuts(xa)) ++xa;
        while (xb >= xa && !cuts(xb)) --xb;
        if (xa > xb) return;
        while (xa > lo && cuts(xa - 1)) --xa;
        while (xb < hi && cuts(xb + 1)) ++xb;
    }
    bool overflow = false;
    uint2* const row = C.slots + ((long long)rz * P.ny + ry) * P.nx;
    for (int x0 = xa; x0 <= xb; x0 += RASTER_BATCH) {
        uint32_t was[RASTER_BATCH];
        int rxs[RASTER_BATCH];
#pragma unroll
        for (int b = 0; b < RASTER_BATCH; ++b) {                                   // independent atomics, issued together
            int rx = x0 + b;
            bool ok = rx <= xb;
            if (P.bc[0]) ok = ok && rx >= 0 && rx < P.nx;
            else rx = rx < 0 ? rx + P.nx : (rx >= P.nx ? rx - P.nx : rx);
            rxs[b] = rx;
            was[b] = ok ? atomicMin(&row[rx].x, (uint32_t)k) : PSM_EMPTY;
        }
#pragma unroll
        for (int b = 0; b < RASTER_BATCH; ++b)
            if (was[b] != PSM_EMPTY && atomicMin(&row[rxs[b]].y, max(was[b], (uint32_t)k)) != PSM_EMPTY) overflow = true;
    }
    if (overflow) atomicOr(C.status, LEDDS_ST_SOLID_OVERFLOW);
}

// ------------------------------------------------------------------------------------ collide + stream
// One block per 128-cell row segment.  The 19 populations of a cell go from global memory straight into the
// thread's column of shared memory with asynchronous copies (no registers tied up while they are in flight);
// the moments are summed from there and the collision runs pair by pair, each pair pushed as soon as it is
// collided.  The kernel needs <= 64 registers, so 8 blocks (32 warps) are resident per SM.
// T = population type: double on the path of the configs; float = the fp32 variant (ledds_coupled_step_f32), where
// the populations, their moments, the collision and the per-cell terms of the solids (Eq. 35-36, 39-42) are single
// precision; which cells a solid cuts is decided by the raster (in double) and the sums of Eq. (41)-(42) over the
// cells are accumulated in double / fixed point as for T = double.
template <typename T, typename I, int BX, bool TRT, bool SUBDIV>
__global__ void __launch_bounds__(PSM_BLOCK, sizeof(T) == 4 ? PSM_MIN_BLOCKS_F32 : PSM_MIN_BLOCKS) lbm_psm_kernel(const T* __restrict__ fin, T* __restrict__ fout,
                                                               const __grid_constant__ LbmDev P,
                                                               const __grid_constant__ CplDev C)
{
    __shared__ T sfull[LEDDS_Q][PSM_BLOCK];
    __shared__ T s2[PSM_S2_ROWS][PSM_BLOCK];
    const int x = blockIdx.x * BX + (int)(threadIdx.x % BX);
    const int y = blockIdx.y * (PSM_BLOCK / BX) + (int)(threadIdx.x / BX), z = blockIdx.z;   // a warp lies inside one row
    const bool active = x < P.nx && y < P.ny;
    const I cell = active ? ((I)z * (I)P.ny + (I)y) * (I)P.nx + (I)x : (I)0;   // a lane past the lattice reads cell 0, stores nothing
    T* sf = &sfull[0][threadIdx.x];
    {
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(sf);
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q)
            asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst + (uint32_t)(q * PSM_BLOCK * sizeof(T))),
                         "l"(fin + (I)((I)q * (I)P.N + cell)), "n"((int)sizeof(T))
                         : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    uint32_t id0 = PSM_EMPTY, id1 = PSM_EMPTY;
    if (active) {
        const uint2 slot = C.slots[cell];
        id0 = slot.x; id1 = slot.y;
    }
    const LbPush<I> push(P, x, y, z);                                                 // index work while the populations are in flight
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    T rho, ux, uy, uz;
    {
        T f[LEDDS_Q];
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) f[q] = sf[q * PSM_BLOCK];
        lb_moments(f, rho, ux, uy, uz);
    }
    if (!__any_sync(0xffffffffu, id0 != PSM_EMPTY)) {
        bgk_collide_stream<I, TRT>(sf, (T)P.omega, rho, ux, uy, uz, push, fout, P, active);
        return;
    }
    if (id0 != PSM_EMPTY) C.slots[cell] = make_uint2(PSM_EMPTY, PSM_EMPTY);           // consumed: free for the next step
    const bool two = __any_sync(0xffffffffu, id1 != PSM_EMPTY);
    T* s2col = &s2[0][threadIdx.x];
    if (two) {                                                                        // warp-uniform, rarer
        T B1, uk1[3], rec[6];
        int ent;
        psm_solid_terms<SUBDIV>(P, C, x, y, z, id1, rho, ux, uy, uz, B1, uk1, rec, ent);
        s2col[0] = B1;
        s2col[PSM_BLOCK] = T(1) - T(1.5) * (uk1[0] * uk1[0] + uk1[1] * uk1[1] + uk1[2] * uk1[2]);
        s2col[2 * PSM_BLOCK] = uk1[0]; s2col[3 * PSM_BLOCK] = uk1[1]; s2col[4 * PSM_BLOCK] = uk1[2];
        psm_run_reduce(C, id1, ent, rec);
    }
    T B0, uk0[3];
    {
        T rec[6];
        int ent;
        psm_solid_terms<SUBDIV>(P, C, x, y, z, id0, rho, ux, uy, uz, B0, uk0, rec, ent);
        psm_run_reduce(C, id0, ent, rec);
    }
    // a warp all of whose cells are inside the lattice and away from every wall pushes without the per-link wall tests
    if (__all_sync(0xffffffffu, active && push.wmask == 0u)) {
        if (!two) psm_collide_stream<I, TRT, true, true>(sf, (T)P.omega, rho, ux, uy, uz, B0, uk0, false, s2col, push, fout, P, active);
        else psm_collide_stream<I, TRT, true, false>(sf, (T)P.omega, rho, ux, uy, uz, B0, uk0, true, s2col, push, fout, P, active);
    } else
        psm_collide_stream<I, TRT, false, false>(sf, (T)P.omega, rho, ux, uy, uz, B0, uk0, two, s2col, push, fout, P, active);
}

template <typename T, typename I, bool TRT, bool SUBDIV>
static void psm_launch2(const T* src, T* dst, const LbmDev& d, const CplDev& C, cudaStream_t st)
{
    const int bx = lb_block_x(d.nx), rows = PSM_BLOCK / bx;
    const dim3 block(PSM_BLOCK), grid((d.nx + bx - 1) / bx, (d.ny + rows - 1) / rows, d.nz);
    if (bx == 128) lbm_psm_kernel<T, I, 128, TRT, SUBDIV><<<grid, block, 0, st>>>(src, dst, d, C);
    else if (bx == 64) lbm_psm_kernel<T, I, 64, TRT, SUBDIV><<<grid, block, 0, st>>>(src, dst, d, C);
    else lbm_psm_kernel<T, I, 32, TRT, SUBDIV><<<grid, block, 0, st>>>(src, dst, d, C);
}

template <typename T, typename I, bool TRT>
static void psm_launch(const T* src, T* dst, const LbmDev& d, const CplDev& C, cudaStream_t st)
{
    if (C.subdiv) psm_launch2<T, I, TRT, true>(src, dst, d, C, st);
    else psm_launch2<T, I, TRT, false>(src, dst, d, C, st);
}

// ------------------------------------------------------------------------------------ finish
// One thread per (solid, component): fixed point -> double, lattice -> DEM units, accumulator reset.
__global__ void cpl_finish_kernel(const CplDev C, double* __restrict__ f_hyd, double* __restrict__ m_hyd)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t == 0) C.blist[0] = 0u;                                                     // the subdivision list is worked through
    if (t >= 6 * C.n) return;
    const int k = t / 6, c = t - 6 * k;
    unsigned long long* a = C.acc + (size_t)t * 2;
    const double v = (double)(long long)a[0] * (1.0 / PSM_FIX_HI) + (double)(long long)a[1] * (1.0 / PSM_FIX_HI / PSM_FIX_LO);
    a[0] = 0ull; a[1] = 0ull;
    if (c < 3) f_hyd[3 * k + c] = v * C.fscale;
    else m_hyd[3 * k + c - 3] = v * C.mscale;
}

// ------------------------------------------------------------------------------------ host API
struct CplLayout { size_t slots, sol, acc, blist, betabox, total; };

static size_t cpl_align(size_t v) { return (v + 255) & ~(size_t)255; }

static int cpl_setup(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c, double r_max, CplDev* C,
                     CplLayout* L)
{
    if (!lbm || !dem || !c || c->n_sub < 1 || (c->solid_fraction != 0 && c->solid_fraction != 1) || !(c->dx > 0.0) || !(c->rho_f > 0.0) || !(r_max > 0.0))
        return LEDDS_EINVAL;
    const double rc = cbrt(3.0 / (4.0 * 3.14159265358979323846));           // Eq. (40), dx = 1
    const double Dt = c->n_sub * dem->d.dt;
    C->n = dem->d.n;
    C->rc = rc;
    C->inv_2rc = 1.0 / (2.0 * rc);
    C->dx = c->dx;
    C->r_max = r_max;
    C->vscale = Dt / c->dx;
    C->wscale = Dt;
    C->fscale = c->rho_f * pow(c->dx, 4) / (Dt * Dt);
    C->mscale = c->rho_f * pow(c->dx, 5) / (Dt * Dt);
    const int nl[3] = {lbm->d.nx, lbm->d.ny, lbm->d.nz};
    C->subdiv = c->solid_fraction ? PSM_NSUB : 0;
    // a cell is cut when its centre is closer than R + r_c (Eq. 40) / when one of its sample points is inside (Eq. 38)
    C->H = (int)ceil(r_max / c->dx + (C->subdiv ? 0.8661 : rc));
    C->S = 2 * C->H + 2;
    if (C->S > 256) return LEDDS_EINVAL;
    for (int a = 0; a < 3; ++a) {
        C->origin[a] = c->origin[a];
        if (dem->d.bc[a] != lbm->d.bc[a]) return LEDDS_EINVAL;              // same topology on both grids
        if (!lbm->d.bc[a] && nl[a] < 2 * C->S) return LEDDS_EINVAL;         // unambiguous nearest image (G33)
    }
    const size_t N = (size_t)lbm->d.N;
    L->slots = 0;
    L->sol = cpl_align(N * sizeof(uint2));
    L->acc = L->sol + cpl_align((size_t)C->n * 10 * sizeof(double));
    const size_t box = (size_t)C->n * C->S * C->S * C->S;
    if (C->subdiv && box >= 0xffffffffull) return LEDDS_EINVAL;
    L->blist = L->acc + cpl_align((size_t)C->n * 12 * sizeof(unsigned long long));      // zeroed with acc at init
    L->betabox = L->blist + (C->subdiv ? cpl_align((box + 1) * sizeof(uint32_t)) : 256);
    L->total = L->betabox + (C->subdiv ? cpl_align(box * sizeof(double)) : 0);
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
        cudaMemsetAsync(base + L.acc, 0, L.blist + 256 - L.acc, st) != cudaSuccess)         // accumulators, list count
        return LEDDS_ECUDA;
    return LEDDS_OK;
}

template <typename T>
static int coupled_step_t(ledds_lbm* lbm, ledds_dem* dem, const ledds_cpl_params* c, double r_max, T* f, double* x, double* v,
                          double* w, double* a, double* alpha, const double* radius, double* f_hyd, double* m_hyd,
                          void* history, void* scratch, void* cpl_scratch, int32_t* status, int nsteps, void* stream)
{
    if (!lbm || !dem || !f || !cpl_scratch || !status || nsteps < 0) return LEDDS_EINVAL;
    if (lbm->f32 != (sizeof(T) == 4)) return LEDDS_EINVAL;                    // the handle fixes the population type
    if (dem->f32) return LEDDS_EINVAL;                                        // the coupled step drives the fp64 DEM
    if (dem->d.n != 0 && (!x || !v || !w || !a || !alpha || !radius || !f_hyd || !m_hyd || !history || !scratch))
        return LEDDS_EINVAL;                                                 // an empty particle system needs none of them
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
    C.hx = reinterpret_cast<const double4*>(sc + s.hx);
    C.pvw = reinterpret_cast<const double*>(sc + s.pvw);
    C.hid = reinterpret_cast<const uint32_t*>(sc + s.hid);
    C.slots = reinterpret_cast<uint2*>(cs + L.slots);
    C.sol = reinterpret_cast<double*>(cs + L.sol);
    C.acc = reinterpret_cast<unsigned long long*>(cs + L.acc);
    C.betabox = C.subdiv ? reinterpret_cast<double*>(cs + L.betabox) : nullptr;
    C.blist = reinterpret_cast<uint32_t*>(cs + L.blist);
    C.status = status;
    const LbmDev& d = lbm->d;
    const size_t half = (size_t)LEDDS_Q * d.N;
    if (d.ny > 65535 || d.nz > 65535) return LEDDS_EINVAL;
    // A kick (with F_sf, M_sf as they stand when it runs) rides on the drift kernel of the next DEM (sub-)step:
    // between sub-steps the values of the previous LBM step are held, and the kick that closes an LBM step
    // rides on the first drift of the next one; only the last step of the call kicks on its own.
    const DemKick hyd = {f_hyd, m_hyd};
    bool pending = false;
    if (nsteps > 0) {                                                        // the DEM state in home order for the whole call
        rc = ledds_dem_import(dem, x, v, w, a, alpha, radius, history, scratch, st);
        if (rc) return rc;
    }
    for (int step = 0; step < nsteps; ++step) {
        for (int sub = 0; sub < c->n_sub; ++sub) {
            // the contact pipeline of the last sub-step runs beside the lattice kernels: only the kick needs both
            const bool fork = sub == c->n_sub - 1 && dem->d.n > 0;
            rc = ledds_dem_advance_contacts(dem, history, scratch, status, dem->d.dt, true, st, fork, pending ? &hyd : nullptr);
            if (rc) return rc;
            pending = sub < c->n_sub - 1;                                    // F_sf of the previous LBM step is held
            if (pending) dem->steps++;
        }
        ledds_prof_start(LEDDS_K_CPL_RASTER, st);
        if (C.n > 0) {
            cpl_solid_kernel<<<(C.n + 127) / 128, 128, 0, st>>>(C);
            ledds_count_launch(1);
            const unsigned rb = (unsigned)(((long long)C.n * C.S * C.S + 255) / 256);
            if (C.subdiv) {
                cpl_beta_classify_kernel<<<(unsigned)(((long long)C.n * C.S * C.S + 255) / 256), 256, 0, st>>>(C);
                cpl_beta_count_kernel<<<ledds_sm_count() * 6, 256, 0, st>>>(C);
                ledds_count_launch(2);
                cpl_raster_kernel<true><<<rb, 256, 0, st>>>(d, C);
            }
            else cpl_raster_kernel<false><<<rb, 256, 0, st>>>(d, C);
        }
        ledds_prof_stop(LEDDS_K_CPL_RASTER, st);
        LEDDS_CHECK_LAUNCH();
        ledds_prof_start(LEDDS_K_LBM, st);
        {
            const T* src = f + lbm->parity * half;
            T* dst = f + (1 - lbm->parity) * half;
            const bool u32 = lb_fits_u32(d.N) && lbm->p.variant != 3;
            if (u32 && !d.trt) psm_launch<T, unsigned, false>(src, dst, d, C, st);
            else if (u32) psm_launch<T, unsigned, true>(src, dst, d, C, st);
            else if (!d.trt) psm_launch<T, long long, false>(src, dst, d, C, st);
            else psm_launch<T, long long, true>(src, dst, d, C, st);
        }
        ledds_prof_stop(LEDDS_K_LBM, st);
        LEDDS_CHECK_LAUNCH();
        lbm->parity ^= 1;
        lbm->steps++;
        ledds_prof_start(LEDDS_K_CPL_REDUCE, st);
        if (C.n > 0) cpl_finish_kernel<<<(6 * C.n + 127) / 128, 128, 0, st>>>(C, f_hyd, m_hyd);
        ledds_prof_stop(LEDDS_K_CPL_REDUCE, st);
        LEDDS_CHECK_LAUNCH();
        if (dem->d.n > 0 && cudaStreamWaitEvent(st, dem->ev_join, 0) != cudaSuccess) return LEDDS_ECUDA;   // join
        dem->steps++;
        pending = step < nsteps - 1;
        if (!pending) {
            rc = ledds_dem_kick(dem, f_hyd, m_hyd, history, scratch, st);
            if (!rc) rc = ledds_dem_export(dem, x, v, w, a, alpha, scratch, st);
            if (rc) return rc;
        }
    }
    return LEDDS_OK;
}

extern "C" int ledds_coupled_step(ledds_lbm* lbm, ledds_dem* dem, const ledds_cpl_params* c, double r_max, double* f,
                                  double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                                  double* f_hyd, double* m_hyd, void* history, void* scratch, void* cpl_scratch,
                                  int32_t* status, int nsteps, void* stream)
{
    return coupled_step_t<double>(lbm, dem, c, r_max, f, x, v, w, a, alpha, radius, f_hyd, m_hyd, history, scratch, cpl_scratch,
                                  status, nsteps, stream);
}

extern "C" int ledds_coupled_step_f32(ledds_lbm* lbm, ledds_dem* dem, const ledds_cpl_params* c, double r_max, float* f,
                                      double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                                      double* f_hyd, double* m_hyd, void* history, void* scratch, void* cpl_scratch,
                                      int32_t* status, int nsteps, void* stream)
{
    return coupled_step_t<float>(lbm, dem, c, r_max, f, x, v, w, a, alpha, radius, f_hyd, m_hyd, history, scratch, cpl_scratch,
                                 status, nsteps, stream);
}
