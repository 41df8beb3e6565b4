// DEM contact pipeline for spheres on sm_100a (Eq. 1-15, 158-192 Eq. 18-21, 431-511).
//
//   dem_drift_key_kernel   Eq. (18a) + predictor, cell key of every particle          (map N_part)
//   dem_hist_kernel        digit histograms of all radix passes in one sweep          (smem histograms)
//   dem_onesweep_kernel    one stable 8-bit radix pass: per-warp match ranking, chained scan with
//                          decoupled look-back across tiles, scatter                    (x passes)
//   dem_gather_kernel      sorted copies of x, v^p, w^p, R + cell start/end from key changes
//   dem_contact_kernel     27-cell walk, Eq. (2)/(6) test, spring-dashpot + Coulomb + torque per pair,
//                          history carried in per-particle slots, per-particle sums in registers
//   dem_kick_kernel        Eq. (18b-c), (19c-d) for spheres
//
// Compiled with -fmad=false: the discrete decisions (cell index, delta_n > 0) must not depend on
// FMA contraction, and none of these kernels is ALU-bound.  No Thrust/CUB; no global fp atomics.
#include <math.h>

#include <new>

#include "common.cuh"

#define DEM_PI 3.14159265358979323846
#define SORT_THREADS 256
#define SORT_WARPS (SORT_THREADS / 32)
#ifndef SORT_ITEMS
#define SORT_ITEMS 12
#endif
#ifndef SORT_MIN_BLOCKS
#define SORT_MIN_BLOCKS 4
#endif
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
#define SORT_RADIX 256

#define ST_FLAG_AGG 0x40000000u
#define ST_FLAG_PRE 0x80000000u
#define ST_VALUE_MASK 0x3fffffffu
#define LOOKBACK 8

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

__device__ __forceinline__ double dem_mass(const DemDev& P, double R) { return P.density * (4.0 / 3.0) * DEM_PI * R * R * R; }

// ------------------------------------------------------------------------------ drift + key
__device__ __forceinline__ int dem_cell_coord(const DemDev& P, double x, int a)
{
    int c = (int)floor((x - P.lo[a]) * P.inv_h[a]);
    c = c < 0 ? 0 : c;
    return c > P.nc[a] - 1 ? P.nc[a] - 1 : c;
}

// Block = DRIFT_BLOCK particles.  The [n][3] arrays are walked as flat arrays (element e = 3 i + k), so every
// load and store is fully coalesced; the new positions pass through shared memory to form the key and the
// packed record per particle.
// KICK = true: the kick of the previous step (Eq. 18b-c, 19c-d with the contact record ft and the external
// force / torque) is applied first, in the same pass: between two steps of one call the state is read and
// written once instead of twice.
#define DRIFT_BLOCK 128
template <bool KICK>
__global__ void __launch_bounds__(DRIFT_BLOCK) dem_drift_key_kernel(
    const DemDev P, double* __restrict__ x, double* __restrict__ v, double* __restrict__ w, double* __restrict__ a,
    double* __restrict__ alpha, const double* __restrict__ radius, const double* __restrict__ ft,
    const double* __restrict__ f_ext, const double* __restrict__ m_ext, double* __restrict__ vp,
    double* __restrict__ wp, double4* __restrict__ xr, uint32_t* __restrict__ key, uint32_t* __restrict__ idx, int drift,
    int32_t* __restrict__ status)
{
    __shared__ double sx[3 * DRIFT_BLOCK];
    const long long e0 = (long long)blockIdx.x * (3 * DRIFT_BLOCK), ne = 3ll * P.n;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int le = threadIdx.x + j * DRIFT_BLOCK;
        const long long e = e0 + le;
        if (e >= ne) break;
        const int k = le % 3;                                                 // e0 is a multiple of 3
        double xv = x[e];
        double vv = v[e], wv = w[e], av = a[e], alv = alpha[e];
        if (KICK) {                                                           // same expressions as dem_kick_kernel
            const int i = (int)(e / 3);
            const double R = radius[i];
            const double m = dem_mass(P, R), I = 0.4 * m * R * R;             // Eq. (21a)
            const double Fq = ft[8 * (size_t)i + k] + (f_ext ? f_ext[e] : 0.0), Mq = ft[8 * (size_t)i + 3 + k] + (m_ext ? m_ext[e] : 0.0);
            const double an = Fq / m + P.g[k], aln = Mq / I;                  // Eq. (18b), (19c)
            vv = vv + (0.5 * P.dt) * (av + an);                               // Eq. (18c)
            wv = wv + (0.5 * P.dt) * (alv + aln);                             // Eq. (19d)
            av = an; alv = aln;
            v[e] = vv; w[e] = wv; a[e] = av; alpha[e] = alv;
        }
        if (drift) {
            xv = xv + P.dt * vv + (0.5 * P.dt * P.dt) * av;                   // Eq. (18a)
            if (!P.bc[k]) {
                if (xv >= P.hi[k]) xv -= P.L[k];
                else if (xv < P.lo[k]) xv += P.L[k];
            }
            x[e] = xv;
            vp[e] = vv + (0.5 * P.dt) * av;                                   // predictor (G11)
            wp[e] = wv + (0.5 * P.dt) * alv;
        } else {
            vp[e] = vv;
            wp[e] = wv;
        }
        sx[le] = xv;
    }
    __syncthreads();
    const int i = blockIdx.x * DRIFT_BLOCK + threadIdx.x;
    if (i >= P.n) return;
    const double xn[3] = {sx[3 * threadIdx.x], sx[3 * threadIdx.x + 1], sx[3 * threadIdx.x + 2]};
    const int cx = dem_cell_coord(P, xn[0], 0), cy = dem_cell_coord(P, xn[1], 1), cz = dem_cell_coord(P, xn[2], 2);
    key[i] = (uint32_t)(cx + P.nc[0] * (cy + P.nc[1] * cz));
    idx[i] = (uint32_t)i;
    const double R = radius[i];
    xr[i] = make_double4(xn[0], xn[1], xn[2], R);                  // one 32-byte sector per particle for the gather
    // input contract (include/ledds.h): 2 R <= cell width, centres inside a walled box
    int st = 2.0 * R > P.hmin ? LEDDS_ST_RADIUS_RANGE : 0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (P.bc[a] && !(xn[a] >= P.lo[a] && xn[a] <= P.hi[a])) st |= LEDDS_ST_OUT_OF_BOX;
    if (st) atomicOr(status, st);
}

// ------------------------------------------------------------------------------ radix sort
// All digit histograms in one pass over the keys (smem atomics, then one global add per bin).
__global__ void __launch_bounds__(SORT_THREADS) dem_hist_kernel(const uint32_t* __restrict__ key, int n, int passes,
                                                               uint32_t* __restrict__ ghist)
{
    __shared__ uint32_t h[4][SORT_RADIX];
    for (int t = threadIdx.x; t < 4 * SORT_RADIX; t += blockDim.x) (&h[0][0])[t] = 0;
    __syncthreads();
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint32_t k = key[i];
        for (int p = 0; p < passes; ++p) atomicAdd(&h[p][(k >> (8 * p)) & 255u], 1u);
    }
    __syncthreads();
    for (int t = threadIdx.x; t < passes * SORT_RADIX; t += blockDim.x) {
        const uint32_t c = (&h[0][0])[t];
        if (c) atomicAdd(&ghist[t], c);
    }
}

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v) { *reinterpret_cast<volatile uint32_t*>(p) = v; }

// One stable LSD pass (8-bit digit at `shift`).  Tiles take tickets from an atomic counter so that
// every tile a block waits on is already resident or done.  Order inside a tile = (warp, item, lane)
// = ascending input index, which keeps the sort stable.
__global__ void __launch_bounds__(SORT_THREADS, SORT_MIN_BLOCKS) dem_onesweep_kernel(
    const uint32_t* __restrict__ key_in, const uint32_t* __restrict__ val_in, uint32_t* __restrict__ key_out,
    uint32_t* __restrict__ val_out, int n, int shift, const uint32_t* __restrict__ ghist /*[256] of this pass*/,
    uint32_t* __restrict__ tile_state /*[tiles][256] of this pass*/, uint32_t* __restrict__ ticket)
{
    __shared__ uint32_t warp_hist[SORT_WARPS][SORT_RADIX];
    __shared__ uint32_t bin_base[SORT_RADIX];
    __shared__ uint32_t tile_start[SORT_RADIX];
    __shared__ uint32_t wsum2[SORT_WARPS];
    __shared__ uint32_t stage_key[SORT_TILE], stage_val[SORT_TILE];
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int t = tid; t < SORT_WARPS * SORT_RADIX; t += SORT_THREADS) (&warp_hist[0][0])[t] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;

    // exclusive prefix of the global digit histogram (thread d owns digit d)
    uint32_t digit_excl;
    {
        const uint32_t c = ghist[tid];
        uint32_t incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        __shared__ uint32_t wsum[SORT_WARPS];
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t base = 0;
        for (int w2 = 0; w2 < warp; ++w2) base += wsum[w2];
        digit_excl = base + incl - c;
    }

    // load (warp-striped) and rank inside the warp
    uint32_t k[SORT_ITEMS], v[SORT_ITEMS], r[SORT_ITEMS];
    const long long base = (long long)tile * SORT_TILE + (long long)warp * (SORT_ITEMS * 32);
#pragma unroll
    for (int it = 0; it < SORT_ITEMS; ++it) {                   // all loads first: 2 x SORT_ITEMS independent requests
        const long long i = base + it * 32 + lane;
        const bool ok = i < n;
        k[it] = ok ? key_in[i] : 0xffffffffu;
        v[it] = ok ? val_in[i] : 0u;
    }
#pragma unroll
    for (int it = 0; it < SORT_ITEMS; ++it) {
        const bool ok = base + it * 32 + lane < n;
        const uint32_t d = ok ? ((k[it] >> shift) & 255u) : 256u;
        uint32_t peers = 0xffffffffu;                               // lanes with the same digit: 9 ballots, one per bit
#pragma unroll
        for (int b = 0; b < 9; ++b) {
            const bool bit = (d >> b) & 1u;
            const uint32_t bal = __ballot_sync(0xffffffffu, bit);
            peers &= bit ? bal : ~bal;
        }
        const uint32_t below = __popc(peers & ((1u << lane) - 1u));
        uint32_t old = 0;
        if (ok) old = warp_hist[warp][d];
        __syncwarp();
        if (ok && below == 0) warp_hist[warp][d] = old + __popc(peers);
        __syncwarp();
        r[it] = old + below;
    }
    __syncthreads();

    // per digit: exclusive scan over the warps of this tile, then the chained scan over tiles
    {
        const int d = tid;
        uint32_t run = 0;
#pragma unroll
        for (int w2 = 0; w2 < SORT_WARPS; ++w2) {
            const uint32_t c = warp_hist[w2][d];
            warp_hist[w2][d] = run;
            run += c;
        }
        uint32_t* my = tile_state + (size_t)tile * SORT_RADIX + d;
        uint32_t excl = 0;
        if (tile == 0) {
            st_volatile(my, ST_FLAG_PRE | run);
        } else {
            st_volatile(my, ST_FLAG_AGG | run);
            // look back over the predecessors' descriptors, LOOKBACK of them per round trip
            long long t = (long long)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t sv[LOOKBACK];
#pragma unroll
                for (int b = 0; b < LOOKBACK; ++b)
                    sv[b] = t - b >= 0 ? ld_volatile(tile_state + (size_t)(t - b) * SORT_RADIX + d) : ST_FLAG_PRE;
#pragma unroll
                for (int b = 0; b < LOOKBACK; ++b) {
                    if (done) break;
                    uint32_t sb = sv[b];
                    while ((sb & (ST_FLAG_AGG | ST_FLAG_PRE)) == 0) sb = ld_volatile(tile_state + (size_t)(t - b) * SORT_RADIX + d);
                    excl += sb & ST_VALUE_MASK;
                    if (sb & ST_FLAG_PRE) done = true;
                }
                t -= LOOKBACK;
            }
            st_volatile(my, ST_FLAG_PRE | (excl + run));
        }
        // where digit d starts inside this tile once the tile is ordered by digit (block-wide exclusive scan of run)
        uint32_t incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) wsum2[warp] = incl;
        __syncthreads();
        uint32_t before = 0;
        for (int w2 = 0; w2 < warp; ++w2) before += wsum2[w2];
        tile_start[d] = before + incl - run;
        bin_base[d] = digit_excl + excl - (before + incl - run);    // global position = bin_base[d] + position in the tile
    }
    __syncthreads();

    // order the tile by digit in shared memory, so that the global writes of a digit are contiguous
#pragma unroll
    for (int it = 0; it < SORT_ITEMS; ++it) {
        if (base + it * 32 + lane < n) {
            const uint32_t d = (k[it] >> shift) & 255u;
            const uint32_t lp = tile_start[d] + warp_hist[warp][d] + r[it];
            stage_key[lp] = k[it];
            stage_val[lp] = v[it];
        }
    }
    __syncthreads();
    const long long tile_first = (long long)tile * SORT_TILE;
    const int count = (int)min((long long)SORT_TILE, (long long)n - tile_first);
    for (int i = tid; i < count; i += SORT_THREADS) {
        const uint32_t kk = stage_key[i];
        const uint32_t dst = bin_base[(kk >> shift) & 255u] + (uint32_t)i;
        key_out[dst] = kk;
        val_out[dst] = stage_val[i];
    }
}

// ------------------------------------------------------------------------------ gather + cell ranges
__global__ void dem_gather_kernel(const DemDev P, const uint32_t* __restrict__ skey, const uint32_t* __restrict__ sidx,
                                  const double4* __restrict__ xr, double4* __restrict__ xr_s,
                                  float4* __restrict__ xf_s, uint2* __restrict__ cell_range)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool ok = s < P.n;
    const uint32_t key = ok ? skey[s] : 0xffffffffu;
    // neighbours' keys inside the warp by shuffle, across warps by one extra load
    uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
    uint32_t next = __shfl_down_sync(0xffffffffu, key, 1);
    if (!ok) return;
    if (lane == 0) prev = s > 0 ? skey[s - 1] : 0xffffffffu;
    if (lane == 31 || s == P.n - 1) next = s < P.n - 1 ? skey[s + 1] : 0xffffffffu;
    if (s == 0 || prev != key) cell_range[key].x = (uint32_t)s;                    // [x, y) = the particles of the cell
    if (s == P.n - 1 || next != key) cell_range[key].y = (uint32_t)s + 1u;
    const double2* src = reinterpret_cast<const double2*>(xr + sidx[s]);
    const double2 a = __ldg(src), b = __ldg(src + 1);
    xr_s[s] = make_double4(a.x, a.y, b.x, b.y);
    // single-precision copy (x - lo, R) for the detect kernel's first look at a candidate (dem_near).  A particle
    // further than 2 L from the box corner (or not finite) gets NaN: it passes every first look.
    const double rx = a.x - P.lo[0], ry = a.y - P.lo[1], rz = b.x - P.lo[2];
    const bool sane = fabs(rx) <= 2.0 * P.L[0] && fabs(ry) <= 2.0 * P.L[1] && fabs(rz) <= 2.0 * P.L[2];
    const float qnan = __int_as_float(0x7fc00000);
    xf_s[s] = sane ? make_float4((float)rx, (float)ry, (float)rz, (float)b.y) : make_float4(qnan, qnan, qnan, qnan);
}

// ------------------------------------------------------------------------------ contact law
struct Body { double x[3], v[3], w[3], R; };

__device__ __forceinline__ void cross3(const double* a, const double* b, double* c)
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

// r_i - r_j with the nearest image on periodic axes
__device__ __forceinline__ void dem_min_image(const DemDev& P, const double* xi, const double* xj, double* d)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        d[a] = xi[a] - xj[a];
        if (!P.bc[a]) {
            if (d[a] > 0.5 * P.L[a]) d[a] -= P.L[a];
            else if (d[a] < -0.5 * P.L[a]) d[a] += P.L[a];
        }
    }
}

// Force of one contact in its canonical orientation (i < j, or j = wall), Eq. (4)-(15).
// en, dn: unit normal from j to i and overlap.  dt3: in = previous delta_t, out = new delta_t.
// F = force on i; T = e_n x F_t (torque on a body of radius R is -R T, Eq. 15).
__device__ __forceinline__ void dem_pair_force(const double* en, double dn, const double* vi, const double* wi,
                                               double Ri, const double* vj, const double* wj, double Rj,
                                               double kn, double kt, double gn, double gt, double mu,
                                               double dt_hist, double* dt3, double* F, double* T)
{
    double rw[3], rwxe[3], vrel[3], vt[3], Ft[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) rw[a] = Ri * wi[a] + Rj * wj[a];
    cross3(rw, en, rwxe);
#pragma unroll
    for (int a = 0; a < 3; ++a) vrel[a] = (vi[a] - vj[a]) - rwxe[a];                  // Eq. (11)
    const double vn = vrel[0] * en[0] + vrel[1] * en[1] + vrel[2] * en[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) vt[a] = vrel[a] - vn * en[a];                         // Eq. (12)
    const double fn = kn * dn - gn * vn;                                              // Eq. (10)
    const double dte = dt3[0] * en[0] + dt3[1] * en[1] + dt3[2] * en[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) dt3[a] = (dt3[a] - dte * en[a]) + dt_hist * vt[a];    // Eq. (13)
#pragma unroll
    for (int a = 0; a < 3; ++a) Ft[a] = -kt * dt3[a] - gt * vt[a];                    // Eq. (4)
    const double ft = sqrt(Ft[0] * Ft[0] + Ft[1] * Ft[1] + Ft[2] * Ft[2]), fmax = mu * fabs(fn);
    if (ft > fmax) {                                                                  // Eq. (5)
        const double s = fmax / ft;
#pragma unroll
        for (int a = 0; a < 3; ++a) { Ft[a] *= s; dt3[a] = -(Ft[a] + gt * vt[a]) / kt; }
    }
    cross3(en, Ft, T);
#pragma unroll
    for (int a = 0; a < 3; ++a) F[a] = fn * en[a] + Ft[a];
}

// One thread per particle, in sorted order, two phases so that the lanes of a warp stay together:
//   1. detect: walk the 9 runs of x-adjacent neighbour cells (they are contiguous in the sorted order), test
//      Eq. (2)/(6) on the packed (x, R) records with squared distances (the square root only when the decision
//      is within rounding) after a first look at the single-precision copy, and note the partners' sorted
//      positions in a per-particle list in global memory;
//   2. evaluate: all lanes work through their k-th contact together: Eq. (7), (10)-(13), (5), (15), history.
// History slots: [sorted position of the step][slot] partner id + delta_t as seen from that particle (the partner
// stores the negated vector).  Per-particle sums stay in registers: no atomics.
// Tuning constants (overridable with -D for sweeps; the defaults are the measured best at 4 M spheres):
#ifndef CONTACT_BLOCK
#define CONTACT_BLOCK 128       // threads per block of both kernels (64 / 256: within 1 %)
#endif
#ifndef DETECT_NB
#define DETECT_NB 3             // candidates in flight per iteration of the detect loop
#endif
#ifndef DETECT_MIN_BLOCKS
#define DETECT_MIN_BLOCKS 8     // caps the detect kernel at 64 registers (8 blocks per SM)
#endif
#ifndef FORCE_MIN_BLOCKS
#define FORCE_MIN_BLOCKS 1      // no register cap on the force kernel (caps spill and run slower)
#endif
#define DEM_IDLE 0xffffffffu   // ncand value of a particle the detect kernel has already finished

// Stiffness and damping of one contact.  HERTZ = false: the linear spring-dashpot of the configs, gamma =
// 2 zeta sqrt(k m*) (G5).  HERTZ = true: Hertz-Mindlin: (A.1) k_n = 4/3 Y* sqrt(R* d_n),
// k_t = 8 G* sqrt(R* d_n); (A.3)-(A.4) S_n = 2 Y* sqrt(R* d_n), S_t = 8 G* sqrt(R* d_n); (A.2) gamma =
// 2 sqrt(5/6) zeta sqrt(S m*), zeta = -beta of (A.5).  Y*, G* of (A.6)-(A.7) come from the host (one material).
template <bool HERTZ>
__device__ __forceinline__ void dem_coefficients(double kn0, double kt0, double Ystar, double Gstar, double zeta, double mstar,
                                                 double Rstar, double dn, double& kn, double& kt, double& gn, double& gt)
{
    if (HERTZ) {
        const double sq = sqrt(Rstar * dn);
        kn = (4.0 / 3.0) * Ystar * sq;
        kt = 8.0 * Gstar * sq;
        const double Sn = 2.0 * Ystar * sq, St = 8.0 * Gstar * sq;
        gn = 2.0 * sqrt(5.0 / 6.0) * zeta * sqrt(Sn * mstar);
        gt = 2.0 * sqrt(5.0 / 6.0) * zeta * sqrt(St * mstar);
    } else {
        kn = kn0; kt = kt0;
        gn = 2.0 * zeta * sqrt(kn * mstar); gt = 2.0 * zeta * sqrt(kt * mstar);
    }
}

// one full 64-byte record per particle: contact force, torque, number of contacts and the row of the history
// arrays that holds them (both exact in a double).  The history rows of a step are in that step's SORTED order
// (row = sorted position): neighbouring threads write neighbouring rows, and because a particle's sorted
// position changes little from one step to the next they also read nearly neighbouring rows.
__device__ __forceinline__ void dem_store_ft(double* __restrict__ ft, uint32_t p, const double* F, const double* M, uint32_t count,
                                             uint32_t row)
{
    double2* o = reinterpret_cast<double2*>(ft + 8 * (size_t)p);
    o[0] = make_double2(F[0], F[1]);
    o[1] = make_double2(F[2], M[0]);
    o[2] = make_double2(M[1], M[2]);
    o[3] = make_double2((double)count, (double)row);
}

// First look at a candidate on the 16-byte single-precision records: false only when the pair is certainly apart.
// Stored coordinates are within 2 L of the origin, so each is off by <= L 2^-23, a difference by <= L 2^-22 (+ the
// rounding of L itself on a wrapped axis) and the distance by < 5e-7 L; fmargin = 2^-19 max L = 1.9e-6 L covers
// that four times over and the factor 1.00001 the roundings of the squares.  NaN records compare as "maybe".
template <bool PERIODIC>
__device__ __forceinline__ bool dem_near(const DemDev& P, const float4& a, const float4& b)
{
    float d[3] = {a.x - b.x, a.y - b.y, a.z - b.z};
    if (PERIODIC) {
#pragma unroll
        for (int k = 0; k < 3; ++k)
            if (!P.bc[k]) {
                if (d[k] > 0.5f * P.Lf[k]) d[k] -= P.Lf[k];
                else if (d[k] < -0.5f * P.Lf[k]) d[k] += P.Lf[k];
            }
    }
    const float d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const float lim = (a.w + b.w) + P.fmargin;
    return !(d2 > lim * lim * 1.00001f);
}

// PERIODIC = false: no axis is periodic, the nearest image is the particle itself
template <bool PERIODIC>
__device__ __forceinline__ bool dem_touch(const DemDev& P, const double4& a, const double4& b)
{
    const double xa[3] = {a.x, a.y, a.z}, xb[3] = {b.x, b.y, b.z};
    double d[3] = {xa[0] - xb[0], xa[1] - xb[1], xa[2] - xb[2]};
    if (PERIODIC) dem_min_image(P, xa, xb, d);
    const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const double sr = a.w + b.w, s2 = sr * sr;
    if (d2 > s2 * (1.0 + 1e-14)) return false;
    if (d2 < s2 * (1.0 - 1e-14)) return true;
    return sr - sqrt(d2) > 0.0;                                                       // Eq. (2), (6), strict (G7)
}

// cand[c][s] (c < ncand[s]) = sorted positions of the particles touching the particle at sorted position s
template <bool PERIODIC>
__global__ void __launch_bounds__(CONTACT_BLOCK, DETECT_MIN_BLOCKS) dem_detect_kernel(
    const DemDev P, const uint32_t* __restrict__ skey, const uint32_t* __restrict__ sidx,
    const double4* __restrict__ xr_s, const float4* __restrict__ xf_s, const uint2* __restrict__ cell_range,
    const double* __restrict__ vp, const double* __restrict__ wp, double2* __restrict__ vw_s, uint32_t* __restrict__ ncand_g,
    uint32_t* __restrict__ cand_g, double* __restrict__ ft_new, int32_t* __restrict__ status)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n) return;
    const int maxc = P.maxc;
    const uint32_t key = skey[s];
    const double4 mine = xr_s[s];
    const float4 minef = xf_s[s];
    int st = 0;
    int ncand = 0;

    const int c0 = (int)(key % (uint32_t)P.nc[0]);
    const int c1 = (int)((key / (uint32_t)P.nc[0]) % (uint32_t)P.nc[1]);
    const int c2 = (int)(key / ((uint32_t)P.nc[0] * (uint32_t)P.nc[1]));

    // ---- phase 1: detect
    auto note = [&](uint32_t t) {
        if (ncand < maxc) cand_g[(size_t)ncand * P.n + s] = t;
        else st |= LEDDS_ST_CONTACT_OVERFLOW;
        ncand += ncand < maxc;
    };
    // the 9 runs [t0, t1) of x-adjacent cells (c0-1 .. c0+1 inside the row): all 27 range loads are independent
    // and issued together; an empty cell holds (0, 0), so "first start, last end" needs no special case
    uint32_t t0[9], t1[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) {
        int qz = c2 + (j / 3 - 1), qy = c1 + (j % 3 - 1);
        bool ok = true;
        if (qz < 0 || qz >= P.nc[2]) { if (P.bc[2]) ok = false; else qz = qz < 0 ? qz + P.nc[2] : qz - P.nc[2]; }
        if (qy < 0 || qy >= P.nc[1]) { if (P.bc[1]) ok = false; else qy = qy < 0 ? qy + P.nc[1] : qy - P.nc[1]; }
        const uint2 none = make_uint2(0u, 0u);
        uint2 r0 = none, r1 = none, r2 = none;
        if (ok) {
            const uint2* row = cell_range + (size_t)P.nc[0] * (size_t)(qy + P.nc[1] * qz) + c0;
            r1 = row[0];
            if (c0 > 0) r0 = row[-1];
            if (c0 < P.nc[0] - 1) r2 = row[1];
        }
        const bool e0 = r0.y > r0.x, e1 = r1.y > r1.x, e2 = r2.y > r2.x;
        t0[j] = e0 ? r0.x : (e1 ? r1.x : r2.x);
        t1[j] = e2 ? r2.y : (e1 ? r1.y : r0.y);
    }
#pragma unroll
    for (int j = 0; j < 9; ++j) {
        for (uint32_t t = t0[j]; t < t1[j]; t += DETECT_NB) {                      // DETECT_NB candidates in flight
            uint32_t tt[DETECT_NB];
            float4 fc[DETECT_NB];
            bool nn[DETECT_NB], any = false;
#pragma unroll
            for (int b = 0; b < DETECT_NB; ++b) {
                tt[b] = min(t + (uint32_t)b, t1[j] - 1u);                          // past the end: the last candidate again
                fc[b] = xf_s[tt[b]];                                               // first look in single precision (no branch),
            }
#pragma unroll
            for (int b = 0; b < DETECT_NB; ++b) {
                nn[b] = dem_near<PERIODIC>(P, minef, fc[b]) & ((int)tt[b] != s) & (b == 0 || tt[b] != tt[b > 0 ? b - 1 : 0]);
                any |= nn[b];
            }
            if (any) {                                                             // Eq. (2) in double for the few that pass
#pragma unroll
                for (int b = 0; b < DETECT_NB; ++b)
                    if (nn[b] && dem_touch<PERIODIC>(P, mine, xr_s[tt[b]])) note(tt[b]);
            }
        }
    }
    if (PERIODIC && !P.bc[0] && (c0 == 0 || c0 == P.nc[0] - 1)) {                  // the wrapped cell of a periodic row
        const int wc = c0 == 0 ? P.nc[0] - 1 : 0;
        for (int j = 0; j < 9; ++j) {
            int qz = c2 + (j / 3 - 1), qy = c1 + (j % 3 - 1);
            if (qz < 0 || qz >= P.nc[2]) { if (P.bc[2]) continue; qz = qz < 0 ? qz + P.nc[2] : qz - P.nc[2]; }
            if (qy < 0 || qy >= P.nc[1]) { if (P.bc[1]) continue; qy = qy < 0 ? qy + P.nc[1] : qy - P.nc[1]; }
            const uint2 r = cell_range[(size_t)P.nc[0] * (size_t)(qy + P.nc[1] * qz) + wc];
            for (uint32_t t = r.x; t < r.y; ++t)
                if ((int)t != s && dem_near<PERIODIC>(P, minef, xf_s[t]) && dem_touch<PERIODIC>(P, mine, xr_s[t])) note(t);
        }
    }

    // a particle that touches nothing and has no wall in reach is finished here (the usual case in a dilute
    // state): zero record written, DEM_IDLE tells the force kernel to skip it
    bool near_wall = false;
    const double xm[3] = {mine.x, mine.y, mine.z};
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (P.bc[a] && (xm[a] - P.lo[a] < mine.w || P.hi[a] - xm[a] < mine.w)) near_wall = true;
    if (ncand == 0 && !near_wall) {
        const double zero[3] = {0.0, 0.0, 0.0};
        dem_store_ft(ft_new, sidx[s], zero, zero, 0u, 0u);
        ncand_g[s] = DEM_IDLE;
    } else {
        // predictor velocities of the particles that take part in a contact, in sorted order: the force kernel
        // reads its own and its partners' (v^p, w^p) from neighbouring records instead of by particle id
        const size_t p3 = 3 * (size_t)sidx[s];
        double2* o = vw_s + 3 * (size_t)s;
        o[0] = make_double2(vp[p3], vp[p3 + 1]);
        o[1] = make_double2(vp[p3 + 2], wp[p3]);
        o[2] = make_double2(wp[p3 + 1], wp[p3 + 2]);
        ncand_g[s] = (uint32_t)ncand;
    }
    if (st) atomicOr(status, st);
}

// ---- phase 2: evaluate
template <bool HERTZ>
__global__ void __launch_bounds__(CONTACT_BLOCK, FORCE_MIN_BLOCKS) dem_force_kernel(
    const DemDev P, const uint32_t* __restrict__ sidx, const double4* __restrict__ xr_s,
    const double2* __restrict__ vw_s, const uint32_t* __restrict__ ncand_g, const uint32_t* __restrict__ cand_g,
    const double* __restrict__ ft_prev, const uint32_t* __restrict__ hid_prev, const double* __restrict__ hdt_prev,
    double* __restrict__ ft_new, uint32_t* __restrict__ hid_new, double* __restrict__ hdt_new,
    int32_t* __restrict__ status, double dt_hist)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n) return;
    const int maxc = P.maxc;
    if (ncand_g[s] == DEM_IDLE) return;
    const double4 mine = xr_s[s];
    const int ncand = (int)ncand_g[s];
    int st = 0;
    const uint32_t p = sidx[s];
    Body me;
    me.x[0] = mine.x; me.x[1] = mine.y; me.x[2] = mine.z; me.R = mine.w;
    {
        const double2* r = vw_s + 3 * (size_t)s;
        const double2 a = r[0], b = r[1], c = r[2];
        me.v[0] = a.x; me.v[1] = a.y; me.v[2] = b.x; me.w[0] = b.y; me.w[1] = c.x; me.w[2] = c.y;
    }
    const double m_me = dem_mass(P, me.R);
    const double2 cr = *reinterpret_cast<const double2*>(ft_prev + 8 * (size_t)p + 6);   // (contacts, row) of the last step
    const uint32_t nprev = (uint32_t)cr.x;
    const size_t prow = (size_t)cr.y;
    const uint32_t* pid = hid_prev + prow * maxc;
    const double* pdt = hdt_prev + prow * maxc * 3;
    uint32_t* nid = hid_new + (size_t)s * maxc;
    double* ndt = hdt_new + (size_t)s * maxc * 3;
    double Fs[3] = {0, 0, 0}, Ms[3] = {0, 0, 0};
    uint32_t ncont = 0;

    for (int c = 0; c < ncand; ++c) {
        const uint32_t t = cand_g[(size_t)c * P.n + s];
        const double4 o4 = xr_s[t];
        const uint32_t q = sidx[t];
        Body ot;
        ot.x[0] = o4.x; ot.x[1] = o4.y; ot.x[2] = o4.z; ot.R = o4.w;
        {
            const double2* r = vw_s + 3 * (size_t)t;
            const double2 a = r[0], b = r[1], c = r[2];
            ot.v[0] = a.x; ot.v[1] = a.y; ot.v[2] = b.x; ot.w[0] = b.y; ot.w[1] = c.x; ot.w[2] = c.y;
        }
        const bool me_first = p < q;                                                   // canonical orientation i < j
        const Body& bi = me_first ? me : ot;
        const Body& bj = me_first ? ot : me;
        double d[3];
        dem_min_image(P, bi.x, bj.x, d);
        const double dist = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        const double dn = (bi.R + bj.R) - dist;                                        // Eq. (6)
        if (dist == 0.0) { st |= LEDDS_ST_COINCIDENT; continue; }
        double en[3] = {d[0] / dist, d[1] / dist, d[2] / dist};                        // Eq. (7)
        const double mi = dem_mass(P, bi.R), mj = dem_mass(P, bj.R);
        const double mstar = mi * mj / (mi + mj);                                      // (A.9)
        const double sg = me_first ? 1.0 : -1.0;
        double dt3[3] = {0, 0, 0};                                                     // previous delta_t, canonical
        for (uint32_t h = 0; h < nprev; ++h)
            if (pid[h] == q) {
                dt3[0] = sg * pdt[3 * h]; dt3[1] = sg * pdt[3 * h + 1]; dt3[2] = sg * pdt[3 * h + 2];
                break;
            }
        double F[3], T[3];
        double kn, kt, gn, gt;
        dem_coefficients<HERTZ>(P.kn, P.kt, P.Ystar, P.Gstar, P.zeta, mstar, bi.R * bj.R / (bi.R + bj.R), dn, kn, kt, gn, gt);
        dem_pair_force(en, dn, bi.v, bi.w, bi.R, bj.v, bj.w, bj.R, kn, kt, gn, gt, P.mu, dt_hist, dt3, F, T);
#pragma unroll
        for (int a = 0; a < 3; ++a) { Fs[a] += sg * F[a]; Ms[a] += me.R * (-T[a]); }
        nid[ncont] = q;
        ndt[3 * ncont] = sg * dt3[0]; ndt[3 * ncont + 1] = sg * dt3[1]; ndt[3 * ncont + 2] = sg * dt3[2];
        ++ncont;
    }
    // walls: static infinite particles with a surface velocity
    for (int wl = 0; wl < 6; ++wl) {
        const int ax = wl >> 1, side = wl & 1;
        if (!P.bc[ax]) continue;
        const double dist = side ? P.hi[ax] - me.x[ax] : me.x[ax] - P.lo[ax];
        const double dn = me.R - dist;
        if (!(dn > 0.0)) continue;
        double en[3] = {0, 0, 0};
        en[ax] = side ? -1.0 : 1.0;
        const uint32_t q = (uint32_t)P.n + (uint32_t)wl;
        double dt3[3] = {0, 0, 0};
        for (uint32_t h = 0; h < nprev; ++h)
            if (pid[h] == q) { dt3[0] = pdt[3 * h]; dt3[1] = pdt[3 * h + 1]; dt3[2] = pdt[3 * h + 2]; break; }
        const double vj[3] = {P.vw[wl * 3], P.vw[wl * 3 + 1], P.vw[wl * 3 + 2]}, wj[3] = {0, 0, 0};
        double F[3], T[3];
        double kn, kt, gn, gt;                                                        // the wall: R* = R_i, m* = m_i
        dem_coefficients<HERTZ>(P.kn_w, P.kt_w, P.Ystar_w, P.Gstar_w, P.zeta_w, m_me, me.R, dn, kn, kt, gn, gt);
        dem_pair_force(en, dn, me.v, me.w, me.R, vj, wj, 0.0, kn, kt, gn, gt, P.mu_w, dt_hist, dt3, F, T);
#pragma unroll
        for (int a = 0; a < 3; ++a) { Fs[a] += F[a]; Ms[a] += me.R * (-T[a]); }
        if (ncont < (uint32_t)maxc) {
            nid[ncont] = q;
            ndt[3 * ncont] = dt3[0]; ndt[3 * ncont + 1] = dt3[1]; ndt[3 * ncont + 2] = dt3[2];
            ++ncont;
        } else st |= LEDDS_ST_CONTACT_OVERFLOW;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (!isfinite(Fs[a]) || !isfinite(Ms[a])) st |= LEDDS_ST_NONFINITE;
    dem_store_ft(ft_new, p, Fs, Ms, ncont, (uint32_t)s);
    if (st) atomicOr(status, st);
}

// ------------------------------------------------------------------------------ kick
// One thread per vector component (element e = 3 i + k of the flat [n][3] arrays): coalesced.
__global__ void dem_kick_kernel(const DemDev P, const double* __restrict__ radius, const double* __restrict__ ft,
                                const double* __restrict__ f_ext, const double* __restrict__ m_ext, double* __restrict__ v,
                                double* __restrict__ w, double* __restrict__ a, double* __restrict__ alpha, int only_accel)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= 3ll * P.n) return;
    const int i = (int)(e / 3), k = (int)(e - 3ll * i);
    const double R = radius[i];
    const double m = dem_mass(P, R), I = 0.4 * m * R * R;                             // Eq. (21a)
    const double Fq = ft[8 * (size_t)i + k] + (f_ext ? f_ext[e] : 0.0), Mq = ft[8 * (size_t)i + 3 + k] + (m_ext ? m_ext[e] : 0.0);
    const double an = Fq / m + P.g[k], aln = Mq / I;                                  // Eq. (18b), (19c)
    if (!only_accel) {
        v[e] = v[e] + (0.5 * P.dt) * (a[e] + an);                                     // Eq. (18c)
        w[e] = w[e] + (0.5 * P.dt) * (alpha[e] + aln);                                // Eq. (19d)
    }
    a[e] = an;
    alpha[e] = aln;
}

// ------------------------------------------------------------------------------ query (parity only)
__global__ void dem_pair_count_kernel(int n, int maxc, const double* __restrict__ ft,
                                      const uint32_t* __restrict__ hid, uint32_t* __restrict__ cnt)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    uint32_t c = 0;
    const uint32_t hc = (uint32_t)ft[8 * (size_t)p + 6];
    const size_t row = (size_t)ft[8 * (size_t)p + 7];
    for (uint32_t h = 0; h < hc; ++h) c += hid[row * maxc + h] > (uint32_t)p;
    cnt[p] = c;
}

__global__ void dem_unpack_ft_kernel(int n, const double* __restrict__ ft, double* __restrict__ force, double* __restrict__ torque)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    for (int a = 0; a < 3; ++a) {
        if (force) force[3 * p + a] = ft[8 * (size_t)p + a];
        if (torque) torque[3 * p + a] = ft[8 * (size_t)p + 3 + a];
    }
}

// single-block exclusive scan of cnt[n] into off[n+1]
__global__ void __launch_bounds__(1024) dem_scan_kernel(int n, const uint32_t* __restrict__ cnt, uint32_t* __restrict__ off)
{
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + tid;
        const uint32_t c = i < n ? cnt[i] : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t s = wsum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, s, o);
                if (lane >= o) s += t;
            }
            wsum[lane] = s;
        }
        __syncthreads();
        const uint32_t before = carry + (warp ? wsum[warp - 1] : 0u) + incl - c;
        if (i < n) off[i] = before;
        __syncthreads();
        if (tid == 1023) carry = before + c;
        __syncthreads();
    }
    if (tid == 0) off[n] = carry;
}

__global__ void dem_pair_write_kernel(int n, int maxc, const double* __restrict__ ft,
                                      const uint32_t* __restrict__ hid, const double* __restrict__ hdt,
                                      const uint32_t* __restrict__ off, uint32_t cap, uint32_t* __restrict__ pairs,
                                      double* __restrict__ pair_dt, uint32_t* __restrict__ n_pairs)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p == 0 && n_pairs) *n_pairs = off[n];
    if (p >= n) return;
    uint32_t ids[32], slot[32];
    int c = 0;
    const uint32_t hc = (uint32_t)ft[8 * (size_t)p + 6];
    const size_t row = (size_t)ft[8 * (size_t)p + 7];
    for (uint32_t h = 0; h < hc; ++h) {
        const uint32_t q = hid[row * maxc + h];
        if (q <= (uint32_t)p) continue;
        int k = c++;
        while (k > 0 && ids[k - 1] > q) { ids[k] = ids[k - 1]; slot[k] = slot[k - 1]; --k; }   // insertion sort
        ids[k] = q; slot[k] = h;
    }
    for (int k = 0; k < c; ++k) {
        const uint32_t o = off[p] + k;
        if (o >= cap) break;
        if (pairs) { pairs[2 * o] = (uint32_t)p; pairs[2 * o + 1] = ids[k]; }
        if (pair_dt)
            for (int a = 0; a < 3; ++a) pair_dt[3 * o + a] = hdt[(row * maxc + slot[k]) * 3 + a];
    }
}

// ------------------------------------------------------------------------------ host API
static double dem_zeta_host(double eps)
{
    if (eps >= 1.0) return 0.0;
    const double l = log(eps);
    return -l / sqrt(l * l + DEM_PI * DEM_PI);                                        // -beta of (A.5)
}

static int dem_setup(const ledds_dem_params* p, ledds_dem* h)
{
    if (!p || p->n < 0 || p->max_contacts < 1 || p->max_contacts > 32) return LEDDS_EINVAL;   // n = 0: a valid, empty system
    if (!(p->cell > 0.0) || !(p->dt >= 0.0) || !(p->density > 0.0)) return LEDDS_EINVAL;
    if (p->model == 0 && (!(p->kn > 0.0) || !(p->kt > 0.0) || !(p->kn_w > 0.0) || !(p->kt_w > 0.0))) return LEDDS_EINVAL;
    if (!(p->restitution > 0.0) || !(p->restitution_w > 0.0) || p->mu < 0.0 || p->mu_w < 0.0) return LEDDS_EINVAL;
    h->p = *p;
    DemDev& d = h->d;
    d.n = p->n;
    double ncell = 1.0;
    d.hmin = 1.0e300;
    for (int a = 0; a < 3; ++a) {
        if (!(p->hi[a] > p->lo[a]) || (p->bc[a] != 0 && p->bc[a] != 1)) return LEDDS_EINVAL;
        d.lo[a] = p->lo[a]; d.hi[a] = p->hi[a]; d.L[a] = p->hi[a] - p->lo[a]; d.bc[a] = p->bc[a];
        d.Lf[a] = (float)d.L[a];
        int nc = (int)floor(d.L[a] / p->cell);
        if (nc < 1) nc = 1;
        if (!p->bc[a] && nc < 3) return LEDDS_EINVAL;          // a periodic axis needs >= 3 cells (27-cell walk)
        d.nc[a] = nc;
        d.inv_h[a] = (double)nc / d.L[a];
        d.hmin = fmin(d.hmin, d.L[a] / (double)nc);
        d.g[a] = p->g[a];
        ncell *= nc;
        for (int s = 0; s < 2; ++s)
            for (int c = 0; c < 3; ++c) d.vw[(a * 2 + s) * 3 + c] = p->v_wall[a][s][c];
    }
    if (ncell > 4.0e9) return LEDDS_EINVAL;
    d.ncell = (unsigned)ncell;
    d.fmargin = (float)(fmax(d.L[0], fmax(d.L[1], d.L[2])) / 524288.0);              // 2^-19 max L (dem_near)
    d.dt = p->dt; d.density = p->density;
    d.kn = p->kn; d.kt = p->kt; d.zeta = dem_zeta_host(p->restitution); d.mu = p->mu;
    d.kn_w = p->kn_w; d.kt_w = p->kt_w; d.zeta_w = dem_zeta_host(p->restitution_w); d.mu_w = p->mu_w;
    d.maxc = p->max_contacts;
    d.Ystar = d.Gstar = d.Ystar_w = d.Gstar_w = 0.0;
    if (p->model != 0 && p->model != 1) return LEDDS_EINVAL;
    if (p->model == 1) {                                                              // (A.6), (A.7)
        const double Ei = p->young, ni = p->poisson, Ew = p->young_w, nw = p->poisson_w;
        if (!(Ei > 0.0) || !(Ew > 0.0) || !(ni > -1.0 && ni < 0.5 + 1e-12) || !(nw > -1.0 && nw < 0.5 + 1e-12)) return LEDDS_EINVAL;
        d.Ystar = 1.0 / ((1.0 - ni * ni) / Ei + (1.0 - ni * ni) / Ei);
        d.Gstar = 1.0 / (2.0 * (2.0 - ni) * (1.0 + ni) / Ei + 2.0 * (2.0 - ni) * (1.0 + ni) / Ei);
        d.Ystar_w = 1.0 / ((1.0 - ni * ni) / Ei + (1.0 - nw * nw) / Ew);
        d.Gstar_w = 1.0 / (2.0 * (2.0 - ni) * (1.0 + ni) / Ei + 2.0 * (2.0 - nw) * (1.0 + nw) / Ew);
    }
    int bits = 1;
    while (bits < 32 && (1ull << bits) < (unsigned long long)d.ncell) ++bits;
    h->key_bits = bits;
    h->passes = (bits + 7) / 8;
    h->tiles = (p->n + SORT_TILE - 1) / SORT_TILE;

    const size_t n = (size_t)p->n;
    size_t o = 0;
    DemScratch& s = h->s;
    auto take = [&](size_t bytes) { const size_t at = o; o += align_up(bytes); return at; };
    // zeroed before every sort: histograms, tickets, tile states (kept contiguous)
    s.hist_digit = take(4 * SORT_RADIX * 4);
    s.tile_counter = take(4 * 4);
    s.tile_state = take((size_t)4 * h->tiles * SORT_RADIX * 4);
    // zeroed before every range build
    s.cell_range = take((size_t)d.ncell * 8);
    for (int b = 0; b < 2; ++b) { s.key[b] = take(n * 4); s.idx[b] = take(n * 4); }
    s.xr = take(n * 32); s.xr_s = take(n * 32); s.xf_s = take(n * 16);
    s.ncand = take(n * 4); s.cand = take(n * d.maxc * 4);
    s.vp = take(n * 24); s.wp = take(n * 24); s.vw_s = take(n * 48);
    s.pair_count = take((n + 1) * 4); s.pair_off = take((n + 1) * 4);
    s.total = o;

    DemHistory& hs = h->hs;
    o = 0;
    for (int b = 0; b < 2; ++b) {
        hs.ft[b] = take(n * 64);
        hs.id[b] = take(n * d.maxc * 4);
        hs.dt[b] = take(n * d.maxc * 24);
    }
    hs.total = o;
    h->cur = 0;
    h->sorted_buf = 0;
    h->steps = 0;
    return LEDDS_OK;
}

extern "C" int ledds_dem_workspace_bytes(const ledds_dem_params* p, size_t* scratch_bytes, size_t* history_bytes)
{
    ledds_dem tmp;
    const int rc = dem_setup(p, &tmp);
    if (rc) return rc;
    if (scratch_bytes) *scratch_bytes = tmp.s.total;
    if (history_bytes) *history_bytes = tmp.hs.total;
    return LEDDS_OK;
}

template <typename T>
static T* at(void* base, size_t off) { return reinterpret_cast<T*>(static_cast<char*>(base) + off); }
template <typename T>
static const T* at(const void* base, size_t off) { return reinterpret_cast<const T*>(static_cast<const char*>(base) + off); }

// drift (optional) -> keys -> sort -> gather/ranges -> contacts.  Leaves force/torque in scratch.
int ledds_dem_advance_contacts(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha,
                               const double* radius, void* history, void* scratch, int32_t* status, double dt_hist,
                               bool drift, cudaStream_t st, bool fork, const DemKick* kick)
{
    // kick != nullptr: the kick that closes the previous step (with the contact forces still in ft[cur] and the
    // external force / torque of *kick) is fused into the drift kernel of this one.
    // fork = true: everything after the drift/key kernel is enqueued on the handle's side stream (ordered after
    // that kernel by an event); the caller joins by waiting on h->ev_join before it needs the contact forces.
    const DemDev& d = h->d;
    const DemScratch& s = h->s;
    const int n = d.n, tb = 128, nb = (n + tb - 1) / tb;
    if (n == 0) { h->cur = 1 - h->cur; return LEDDS_OK; }
    // clear sort bookkeeping + cell ranges (one contiguous region)
    if (cudaMemsetAsync(at<char>(scratch, s.hist_digit), 0, s.key[0] - s.hist_digit, st) != cudaSuccess) return LEDDS_ECUDA;
    ledds_prof_start(LEDDS_K_DEM_KEYS, st);
    {
        const dim3 grid((n + DRIFT_BLOCK - 1) / DRIFT_BLOCK);
        const double* ft = at<double>(history, h->hs.ft[h->cur]);
        if (kick)
            dem_drift_key_kernel<true><<<grid, DRIFT_BLOCK, 0, st>>>(d, x, v, w, a, alpha, radius, ft, kick->f_ext, kick->m_ext,
                                                                      at<double>(scratch, s.vp), at<double>(scratch, s.wp), at<double4>(scratch, s.xr),
                                                                      at<uint32_t>(scratch, s.key[0]), at<uint32_t>(scratch, s.idx[0]), drift ? 1 : 0, status);
        else
            dem_drift_key_kernel<false><<<grid, DRIFT_BLOCK, 0, st>>>(d, x, v, w, a, alpha, radius, ft, nullptr, nullptr,
                                                                       at<double>(scratch, s.vp), at<double>(scratch, s.wp), at<double4>(scratch, s.xr),
                                                                       at<uint32_t>(scratch, s.key[0]), at<uint32_t>(scratch, s.idx[0]), drift ? 1 : 0, status);
    }
    ledds_prof_stop(LEDDS_K_DEM_KEYS, st);
    LEDDS_CHECK_LAUNCH();
    if (fork) {
        if (!h->side && (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
                         cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                         cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess))
            return LEDDS_ECUDA;
        if (cudaEventRecord(h->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(h->side, h->ev_fork, 0) != cudaSuccess)
            return LEDDS_ECUDA;
        st = h->side;
    }
    ledds_prof_start(LEDDS_K_DEM_SORT, st);
    int hb = (n + SORT_THREADS * 8 - 1) / (SORT_THREADS * 8);
    if (hb > ledds_sm_count() * 8) hb = ledds_sm_count() * 8;
    dem_hist_kernel<<<hb, SORT_THREADS, 0, st>>>(at<uint32_t>(scratch, s.key[0]), n, h->passes,
                                                 at<uint32_t>(scratch, s.hist_digit));
    LEDDS_CHECK_LAUNCH();
    for (int p = 0; p < h->passes; ++p) {
        const int in = p & 1, out = in ^ 1;
        dem_onesweep_kernel<<<h->tiles, SORT_THREADS, 0, st>>>(
            at<uint32_t>(scratch, s.key[in]), at<uint32_t>(scratch, s.idx[in]), at<uint32_t>(scratch, s.key[out]),
            at<uint32_t>(scratch, s.idx[out]), n, 8 * p, at<uint32_t>(scratch, s.hist_digit) + p * SORT_RADIX,
            at<uint32_t>(scratch, s.tile_state) + (size_t)p * h->tiles * SORT_RADIX,
            at<uint32_t>(scratch, s.tile_counter) + p);
        LEDDS_CHECK_LAUNCH();
    }
    ledds_prof_stop(LEDDS_K_DEM_SORT, st);
    h->sorted_buf = h->passes & 1;
    const uint32_t* skey = at<uint32_t>(scratch, s.key[h->sorted_buf]);
    const uint32_t* sidx = at<uint32_t>(scratch, s.idx[h->sorted_buf]);
    ledds_prof_start(LEDDS_K_DEM_GATHER, st);
    dem_gather_kernel<<<nb, tb, 0, st>>>(d, skey, sidx, at<double4>(scratch, s.xr), at<double4>(scratch, s.xr_s),
                                         at<float4>(scratch, s.xf_s), at<uint2>(scratch, s.cell_range));
    ledds_prof_stop(LEDDS_K_DEM_GATHER, st);
    LEDDS_CHECK_LAUNCH();
    const DemHistory& hs = h->hs;
    const int prev = h->cur, nw = 1 - h->cur;
    ledds_prof_start(LEDDS_K_DEM_CONTACT, st);
    if (d.bc[0] && d.bc[1] && d.bc[2])
        dem_detect_kernel<false><<<(n + CONTACT_BLOCK - 1) / CONTACT_BLOCK, CONTACT_BLOCK, 0, st>>>(d, skey, sidx, at<double4>(scratch, s.xr_s), at<float4>(scratch, s.xf_s), at<uint2>(scratch, s.cell_range),
                                                               at<double>(scratch, s.vp), at<double>(scratch, s.wp), at<double2>(scratch, s.vw_s),
                                                               at<uint32_t>(scratch, s.ncand), at<uint32_t>(scratch, s.cand),
                                                               at<double>(history, hs.ft[nw]), status);
    else
        dem_detect_kernel<true><<<(n + CONTACT_BLOCK - 1) / CONTACT_BLOCK, CONTACT_BLOCK, 0, st>>>(d, skey, sidx, at<double4>(scratch, s.xr_s), at<float4>(scratch, s.xf_s), at<uint2>(scratch, s.cell_range),
                                                              at<double>(scratch, s.vp), at<double>(scratch, s.wp), at<double2>(scratch, s.vw_s),
                                                              at<uint32_t>(scratch, s.ncand), at<uint32_t>(scratch, s.cand),
                                                              at<double>(history, hs.ft[nw]), status);
    ledds_count_launch(1);
    (h->p.model == 1 ? dem_force_kernel<true> : dem_force_kernel<false>)<<<(n + CONTACT_BLOCK - 1) / CONTACT_BLOCK, CONTACT_BLOCK, 0, st>>>(
        d, sidx, at<double4>(scratch, s.xr_s), at<double2>(scratch, s.vw_s),
        at<uint32_t>(scratch, s.ncand), at<uint32_t>(scratch, s.cand),
        at<double>(history, hs.ft[prev]), at<uint32_t>(history, hs.id[prev]), at<double>(history, hs.dt[prev]),
        at<double>(history, hs.ft[nw]), at<uint32_t>(history, hs.id[nw]), at<double>(history, hs.dt[nw]), status, dt_hist);
    ledds_prof_stop(LEDDS_K_DEM_CONTACT, st);
    LEDDS_CHECK_LAUNCH();
    h->cur = nw;
    if (fork && cudaEventRecord(h->ev_join, st) != cudaSuccess) return LEDDS_ECUDA;
    return LEDDS_OK;
}

int ledds_dem_kick(ledds_dem* h, double* v, double* w, double* a, double* alpha, const double* radius,
                   const double* f_ext, const double* m_ext, const void* history, int32_t* status, cudaStream_t st)
{
    (void)status;
    const int n = h->d.n;
    if (n == 0) return LEDDS_OK;
    ledds_prof_start(LEDDS_K_DEM_KICK, st);
    dem_kick_kernel<<<(unsigned)((3ll * n + 255) / 256), 256, 0, st>>>(h->d, radius, at<double>(history, h->hs.ft[h->cur]), f_ext, m_ext, v, w, a, alpha, 0);
    ledds_prof_stop(LEDDS_K_DEM_KICK, st);
    LEDDS_CHECK_LAUNCH();
    return LEDDS_OK;
}

extern "C" int ledds_dem_init(ledds_dem** out, const ledds_dem_params* p, const double* x, const double* v,
                              const double* w, const double* radius, double* a, double* alpha, void* history,
                              void* scratch, int32_t* status, void* stream)
{
    if (!out || !p || !status) return LEDDS_EINVAL;
    if (p->n != 0 && (!x || !v || !w || !radius || !a || !alpha || !history || !scratch)) return LEDDS_EINVAL;
    const void* ptrs[] = {x, v, w, radius, a, alpha, history, scratch, status};
    for (const void* q : ptrs)
        if (!ledds_aligned16(q)) return LEDDS_EALIGN;
    ledds_dem* h = new (std::nothrow) ledds_dem();
    if (!h) return LEDDS_EINVAL;
    int rc = dem_setup(p, h);
    if (rc) { delete h; return rc; }
    cudaStream_t st = (cudaStream_t)stream;
    if ((h->hs.total && cudaMemsetAsync(history, 0, h->hs.total, st) != cudaSuccess) ||
        cudaMemsetAsync(status, 0, 16, st) != cudaSuccess) {
        delete h;
        return LEDDS_ECUDA;
    }
    // forces of the initial state: no drift, delta_t stays 0 (dt_hist = 0)
    rc = ledds_dem_advance_contacts(h, const_cast<double*>(x), const_cast<double*>(v), const_cast<double*>(w), a, alpha, radius, history,
                                    scratch, status, 0.0, false, st, false, nullptr);
    if (rc) { delete h; return rc; }
    if (h->d.n == 0) { *out = h; return LEDDS_OK; }
    dem_kick_kernel<<<(unsigned)((3ll * h->d.n + 255) / 256), 256, 0, st>>>(h->d, radius, at<double>(history, h->hs.ft[h->cur]), nullptr,
                                                                            nullptr, nullptr, nullptr, a, alpha, 1);
    ledds_count_launch(1);
    if (cudaPeekAtLastError() != cudaSuccess) { delete h; return LEDDS_ECUDA; }
    *out = h;
    return LEDDS_OK;
}

extern "C" int ledds_dem_step(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha,
                              const double* radius, const double* f_ext, const double* m_ext, void* history,
                              void* scratch, int32_t* status, int nsteps, void* stream)
{
    if (!h || !status || nsteps < 0) return LEDDS_EINVAL;
    if (h->d.n == 0) return LEDDS_OK;
    if (!x || !v || !w || !a || !alpha || !radius || !history || !scratch) return LEDDS_EINVAL;
    const void* ptrs[] = {x, v, w, a, alpha, radius, f_ext, m_ext, history, scratch, status};
    for (const void* q : ptrs)
        if (!ledds_aligned16(q)) return LEDDS_EALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    const DemKick kick = {f_ext, m_ext};
    for (int s = 0; s < nsteps; ++s) {
        // the kick of step s - 1 rides on the drift of step s; only the last step of the call kicks on its own
        int rc = ledds_dem_advance_contacts(h, x, v, w, a, alpha, radius, history, scratch, status, h->d.dt, true, st, false,
                                            s > 0 ? &kick : nullptr);
        if (rc) return rc;
        h->steps++;
    }
    if (nsteps > 0) return ledds_dem_kick(h, v, w, a, alpha, radius, f_ext, m_ext, history, status, st);
    return LEDDS_OK;
}

extern "C" int ledds_dem_query(ledds_dem* h, const void* history, const void* scratch, uint32_t* sorted_idx,
                               uint32_t* sorted_key, uint32_t* pairs, double* pair_dt, uint32_t pair_cap,
                               uint32_t* n_pairs, double* force, double* torque, void* stream)
{
    if (!h) return LEDDS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)h->d.n;
    if (n == 0) {
        if (n_pairs && cudaMemsetAsync(n_pairs, 0, sizeof(uint32_t), st) != cudaSuccess) return LEDDS_ECUDA;
        return LEDDS_OK;
    }
    if (!history || !scratch) return LEDDS_EINVAL;
    const DemScratch& s = h->s;
    auto copy = [&](void* dst, const void* src, size_t bytes) {
        return !dst || cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, st) == cudaSuccess;
    };
    if (!copy(sorted_idx, at<char>(scratch, s.idx[h->sorted_buf]), n * 4) ||
        !copy(sorted_key, at<char>(scratch, s.key[h->sorted_buf]), n * 4))
        return LEDDS_ECUDA;
    if (force || torque) {
        dem_unpack_ft_kernel<<<((int)n + 127) / 128, 128, 0, st>>>((int)n, at<double>(history, h->hs.ft[h->cur]), force, torque);
        LEDDS_CHECK_LAUNCH();
    }
    if (pairs || pair_dt || n_pairs) {
        const DemHistory& hs = h->hs;
        const int tb = 128, nb = ((int)n + tb - 1) / tb;
        // scratch is logically const for the caller; the two query arrays are ours to overwrite
        uint32_t* cnt = const_cast<uint32_t*>(at<uint32_t>(scratch, s.pair_count));
        uint32_t* off = const_cast<uint32_t*>(at<uint32_t>(scratch, s.pair_off));
        dem_pair_count_kernel<<<nb, tb, 0, st>>>((int)n, h->d.maxc, at<double>(history, hs.ft[h->cur]),
                                                 at<uint32_t>(history, hs.id[h->cur]), cnt);
        dem_scan_kernel<<<1, 1024, 0, st>>>((int)n, cnt, off);
        dem_pair_write_kernel<<<nb, tb, 0, st>>>((int)n, h->d.maxc, at<double>(history, hs.ft[h->cur]),
                                                 at<uint32_t>(history, hs.id[h->cur]), at<double>(history, hs.dt[h->cur]),
                                                 off, pair_cap, pairs, pair_dt, n_pairs);
        ledds_count_launch(2);
        LEDDS_CHECK_LAUNCH();
    }
    return LEDDS_OK;
}

extern "C" int ledds_dem_destroy(ledds_dem* h)
{
    if (h && h->side) {
        cudaStreamDestroy(h->side);
        cudaEventDestroy(h->ev_fork);
        cudaEventDestroy(h->ev_join);
    }
    delete h;
    return LEDDS_OK;
}
