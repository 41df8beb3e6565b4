// Device code of the PSM coupling kernels (Eq. 32-42).  Included by coupled.cu.
#pragma once
#include "lbm_kernels.cuh"

#define PSM_BLOCK 128
#define PSM_MIN_BLOCKS 6      // resident blocks per SM the collide kernel is compiled for (<= 85 registers)
#define PSM_MIN_BLOCKS_F32 8  // the same for float populations (<= 64 registers)
#define PSM_EMPTY 0xffffffffu

// Layout of the caller-owned coupling scratch (ledds_cpl_workspace_bytes):
//   slots[N]            uint2 per fluid cell: the (<= 2, lowest) ids of the solids cutting it, PSM_EMPTY
//                       when free.  Written by cpl_raster_kernel, consumed and reset by lbm_psm_kernel,
//                       so it is all-empty between steps.
//   sol[n][10]          per solid, lattice units: x_k[3], R_k, v_k[3], w_k[3] (predictor values)
//   betabox[n][S^3]     double: solid fraction of Eq. (38) per (solid, cell of its bounding box); only allocated
//                       and used with the subdivision method (written by the raster, read by the collide kernel)
//   acc[n][6][2]        uint64: per solid and component of (F, M), the exact sum of the (cell, solid) terms of
//                       Eq. (41)-(42) in 2^-83 fixed point (two limbs: units of 2^-30 and of 2^-83).  Integer
//                       additions commute, so the sum does not depend on the order in which blocks finish;
//                       cpl_finish_kernel converts and resets it.
struct CplDev {
    int n;
    double rc, inv_2rc;        // Eq. (40) in lattice units
    double dx, vscale, wscale, origin[3];
    double r_max;              // largest radius the scratch and the raster boxes were sized for (DEM units)
    double fscale, mscale;     // lattice -> DEM units for force / torque
    int H, S;                  // half-width and width of the solid's bounding box in cells (raster)
    int subdiv;                // 0: distance-based solid fraction Eq. (39)-(40); else points per direction of Eq. (38)
    double* betabox;           // [n][S^3] solid fraction per (solid, cell of its box), subdivision method only
    uint32_t* blist;           // [0] = count, [1..]: box-cell indices k S^3 + e whose points have to be counted
    const double4* hx; const double* pvw; const uint32_t* hid;   // DEM state in home order: (x, R), predictor (v^p, w^p), particle id
    uint2* slots;
    double* sol;
    unsigned long long* acc;
    int32_t* status;
};

// delta_sc of Eq. (40) > 0, evaluated with explicitly rounded operations so that the raster kernel and
// the collide kernel take the same decision for the same (cell, solid) whatever the compiler contracts.
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

// delta_sc > 0 (Eq. 39-40) decided exactly as cpl_dsc(...) > 0 would, but without the square root unless
// the squared distance is within rounding of (R_k + r_c)^2.
__device__ __forceinline__ bool cpl_cuts(double Rk, double rc, const double* d)
{
    const double s = __dadd_rn(Rk, rc), s2 = s * s;
    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
    if (d2 < s2 * (1.0 - 1e-14)) return true;
    if (d2 > s2 * (1.0 + 1e-14)) return false;
    return __dsub_rn(s, __dsqrt_rn(d2)) > 0.0;
}

// Eq. (38), subdivision method with PSM_NSUB points per direction at r_j + ((a + 1/2)/NSUB - 1/2); d = r_j - r_k.
// Each point is tested as the oracle tests it (explicitly rounded operations), so the count is the same; cells
// whose farthest point is inside / nearest point is outside need no count (rounding is monotone).
#define PSM_NSUB 10
struct SubdivPoints { double s2[3][PSM_NSUB], lo2[3], hi2[3], R2; };

__device__ __forceinline__ void cpl_subdiv_points(const double* d, double Rk, SubdivPoints& p)
{
    p.R2 = __dmul_rn(Rk, Rk);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        p.lo2[a] = 1.0e300; p.hi2[a] = 0.0;
#pragma unroll
        for (int i = 0; i < PSM_NSUB; ++i) {
            const double off = ((double)i + 0.5) / (double)PSM_NSUB - 0.5;           // folded at compile time (IEEE, as the oracle's)
            const double sv = __dadd_rn(d[a], off);
            p.s2[a][i] = __dmul_rn(sv, sv);
            p.lo2[a] = fmin(p.lo2[a], p.s2[a][i]);
            p.hi2[a] = fmax(p.hi2[a], p.s2[a][i]);
        }
    }
}

// 1 / 0 when every / no point is inside, -1 when the points have to be counted
__device__ __forceinline__ double cpl_beta_classify(const SubdivPoints& p)
{
    if (__dadd_rn(__dadd_rn(p.hi2[0], p.hi2[1]), p.hi2[2]) < p.R2) return 1.0;
    if (!(__dadd_rn(__dadd_rn(p.lo2[0], p.lo2[1]), p.lo2[2]) < p.R2)) return 0.0;
    return -1.0;
}

// Number of the NSUB^3 points inside, exactly as the oracle counts them -- (sx^2 + sy^2) + sz^2 < R^2 with every operation
// rounded -- but without testing every point: rounding is monotone, so with the ten squares of the z offsets put in
// ascending order the points of a column (x, y) that pass are a prefix of them, and its length comes from a 4-step
// search instead of 10 tests (the 100 searches are independent: no loop-carried chain).  zs = this thread's column of
// shared memory (stride `zstride` doubles) for the sorted z squares, which the search indexes.
__device__ __forceinline__ void cpl_sort10(double (&v)[PSM_NSUB])
{
#pragma unroll
    for (int r = 0; r < PSM_NSUB; ++r)                                               // odd-even transposition network
#pragma unroll
        for (int i = r & 1; i + 1 < PSM_NSUB; i += 2) {
            const double lo = fmin(v[i], v[i + 1]), hi = fmax(v[i], v[i + 1]);
            v[i] = lo; v[i + 1] = hi;
        }
}

__device__ __forceinline__ double cpl_beta_count(const SubdivPoints& p, double* zs, int zstride)
{
    double z[PSM_NSUB];
#pragma unroll
    for (int i = 0; i < PSM_NSUB; ++i) z[i] = p.s2[2][i];
    cpl_sort10(z);
#pragma unroll
    for (int i = 0; i < PSM_NSUB; ++i) zs[i * zstride] = z[i];
    int count = 0;
#pragma unroll
    for (int a = 0; a < PSM_NSUB; ++a)
#pragma unroll
        for (int b = 0; b < PSM_NSUB; ++b) {
            const double sxy = __dadd_rn(p.s2[0][a], p.s2[1][b]);                   // (sx^2 + sy^2) + sz^2, as the oracle sums
            int pos = 0;                                                             // z squares 0 .. pos-1 pass
#pragma unroll
            for (int step = 8; step > 0; step >>= 1) {
                const int q = pos + step;
                const bool ok = q <= PSM_NSUB && __dadd_rn(sxy, zs[(min(q, PSM_NSUB) - 1) * zstride]) < p.R2;
                pos = ok ? q : pos;
            }
            count += pos;
        }
    return (double)count / (double)(PSM_NSUB * PSM_NSUB * PSM_NSUB);
}

// What one solid does to one cell: weight B (Eq. 36, 39-40), solid velocity at the cell (Eq. 35), the terms
// of Eq. (41)-(42) in lattice units (rec) and the index of the cell in the solid's box (ent).
// id = PSM_EMPTY: no solid here: B = 0, rec = 0, ent = -1 (the lane still runs the code of its warp).
// R = arithmetic type of the cell's terms: double, or float for the fp32 lattice (there the offsets d = r_j - r_k are
// still formed in double from the same floor(x_k) as the raster's, so `ent` addresses the same box cell).
template <bool SUBDIV, typename R>
__device__ __forceinline__ void psm_solid_terms(const LbmDev& P, const CplDev& C, int x, int y, int z, uint32_t id,
                                                R rho, R ux, R uy, R uz, R& B, R (&uk)[3], R (&rec)[6], int& ent)
{
    const bool has = id != PSM_EMPTY;
    const uint32_t k = has ? id : 0u;
    const double2* sp = reinterpret_cast<const double2*>(C.sol + (size_t)k * 10);
    const double2 a0 = __ldg(sp), a1 = __ldg(sp + 1), a2 = __ldg(sp + 2), a3 = __ldg(sp + 3), a4 = __ldg(sp + 4);
    const double xk[3] = {a0.x, a0.y, a1.x}, Rk = a1.y;
    const R vk[3] = {(R)a2.x, (R)a2.y, (R)a3.x}, wk[3] = {(R)a3.y, (R)a4.x, (R)a4.y};
    const int fk[3] = {(int)floor(xk[0]), (int)floor(xk[1]), (int)floor(xk[2])};
    const int di[3] = {cpl_offset(x, fk[0], P.nx, !P.bc[0]), cpl_offset(y, fk[1], P.ny, !P.bc[1]),
                       cpl_offset(z, fk[2], P.nz, !P.bc[2])};
    double dd[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) dd[a] = (double)(fk[a] + di[a]) - xk[a];             // r_j - r_k, nearest image
    const R d[3] = {(R)dd[0], (R)dd[1], (R)dd[2]};
    ent = has ? ((di[2] + C.H) * C.S + (di[1] + C.H)) * C.S + (di[0] + C.H) : -1;
    R beta;
    if (SUBDIV) {
        beta = has ? (R)C.betabox[(size_t)k * (size_t)(C.S * C.S * C.S) + (size_t)ent] : R(0);   // Eq. (38), from the raster
    } else {
        if constexpr (sizeof(R) == 8) {
            const double dsc = cpl_dsc(Rk, C.rc, cpl_dist(dd));
            beta = dsc * C.inv_2rc;                                                  // Eq. (39)-(40)
        } else {
            const float dist = __fsqrt_rn(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            beta = (((float)Rk + (float)C.rc) - dist) * (float)C.inv_2rc;
        }
        beta = beta > R(1) ? R(1) : beta;
        beta = (has && beta > R(0)) ? beta : R(0);
    }
    const R tm = (R)(P.tau - 0.5);
    {   // Eq. (36).  A lane without a solid (beta = 0) divides a stand-in value instead of 0: a zero numerator sends the
        // whole warp through the slow path of the division; the lanes with a solid compute exactly beta tm / (1 - beta + tm)
        const bool on = beta > R(0);
        const R bb = on ? beta : R(0.5);
        const R q = bb * tm / ((R(1) - bb) + tm);
        B = on ? q : R(0);
    }
    uk[0] = vk[0] + (wk[1] * d[2] - wk[2] * d[1]);                                   // Eq. (35)
    uk[1] = vk[1] + (wk[2] * d[0] - wk[0] * d[2]);
    uk[2] = vk[2] + (wk[0] * d[1] - wk[1] * d[0]);
    // Eq. (41): -B_k sum_i Omega^s_{i,k} c_i.  The sum is rho (u_k - u) identically (sum_i c_i f_i = rho u,
    // sum_i c_i f_i^eq(rho, v) = rho v, c_opp = -c), so it is formed from the moments.
    const R Br = B * rho;
    const R dF[3] = {Br * (ux - uk[0]), Br * (uy - uk[1]), Br * (uz - uk[2])};       // lattice units
    rec[0] = dF[0]; rec[1] = dF[1]; rec[2] = dF[2];
    rec[3] = d[1] * dF[2] - d[2] * dF[1];                                            // Eq. (42)
    rec[4] = d[2] * dF[0] - d[0] * dF[2];
    rec[5] = d[0] * dF[1] - d[1] * dF[0];
}

// Second solid of a cell, parked in shared memory while the collision runs (one column per thread):
// rows 0..4 = B, 1 - 1.5 u_k^2, u_k[3].
#define PSM_S2_ROWS 5

// Sum the records of each run of consecutive lanes that hold the same solid id (a solid cuts a lattice row
// in consecutive cells) with a shuffle tree, and let the first lane of the run add the sum to the solid's
// fixed-point accumulators (12 integer reductions, no return value).  All 32 lanes call this; id = PSM_EMPTY
// marks a lane without a record.  ent is unused here (kept for the callers' bookkeeping).
#define PSM_FIX_HI 1073741824.0                /* 2^30 */
#define PSM_FIX_LO 9007199254740992.0          /* 2^53 */
template <typename R>
__device__ __forceinline__ void psm_run_reduce(const CplDev& C, uint32_t id, int ent, R (&v)[6])
{
    (void)ent;
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const uint32_t prev = __shfl_up_sync(full, id, 1);
    const unsigned starts = __ballot_sync(full, lane == 0 || prev != id);          // bit l: lane l begins a run
    const unsigned above = lane == 31 ? 0u : (starts >> (lane + 1));
    const int len = id == PSM_EMPTY ? 1 : (above ? __ffs(above) : 32 - lane);       // lanes from here to the end of my run
    const int maxlen = __reduce_max_sync(full, len);                                // runs are ~2 (R + r_c) cells long
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        if (o >= maxlen) break;
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            const R t = __shfl_down_sync(full, v[c], o);
            if (o < len) v[c] += t;
        }
    }
    if (id != PSM_EMPTY && ((starts >> lane) & 1u)) {
        unsigned long long* a = C.acc + (size_t)id * 12;
        double big = fabs((double)v[0]);                                           // NaN-propagating: fmax would drop a NaN
#pragma unroll
        for (int c = 1; c < 6; ++c) big += fabs((double)v[c]);
        if (!(big < 4.0e9)) { atomicOr(C.status, LEDDS_ST_NONFINITE); return; }
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            const double s = (double)v[c] * PSM_FIX_HI, h = rint(s), l = rint((s - h) * PSM_FIX_LO);   // s - h is exact
            atomicAdd(a + 2 * c, (unsigned long long)(long long)h);
            atomicAdd(a + 2 * c + 1, (unsigned long long)(long long)l);
        }
    }
}

// ---- streaming forms: the populations of the cell sit in shared memory (column `sf`, stride PSM_BLOCK), are
// collided pair by pair and pushed right away, so that only one pair is live in registers at a time.

// BGK or TRT without solids, same expressions as lb_collide_bgk / lb_collide_trt
template <typename I, bool TRT, typename T>
__device__ __forceinline__ void bgk_collide_stream(const T* sf, T omega, T rho, T ux, T uy, T uz,
                                                   const LbPush<I>& push, T* __restrict__ fout, const LbmDev& P, bool active)
{
    if (TRT) {
        const T k = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
        {
            const T f0 = sf[0];
            if (active) push.put(fout, P, 0, f0 - omega * (f0 - T(lb_w(0)) * rho * k), rho);
        }
#pragma unroll
        for (int q = 1; q < LEDDS_Q; q += 2) {
            const T a = sf[q * PSM_BLOCK], b = sf[(q + 1) * PSM_BLOCK];
            const T cu = lb_cdot(q, ux, uy, uz);
            const T wr = T(lb_w(q)) * rho;
            const T even = wr * (k + T(4.5) * cu * cu), odd = wr * T(3) * cu;
            const T rp = omega * (T(0.5) * (a + b) - even), rm = (T)P.omega_minus * (T(0.5) * (a - b) - odd);
            if (active) {
                push.put(fout, P, q, a - (rp + rm), rho);
                push.put(fout, P, q + 1, b - (rp - rm), rho);
            }
        }
        return;
    }
    const T k = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    {
        const T f0 = sf[0], fe = T(lb_w(0)) * rho * k;
        if (active) push.put(fout, P, 0, f0 - omega * (f0 - fe), rho);
    }
#pragma unroll
    for (int q = 1; q < LEDDS_Q; q += 2) {
        const T a = sf[q * PSM_BLOCK], b = sf[(q + 1) * PSM_BLOCK];
        const T cu = lb_cdot(q, ux, uy, uz);
        const T wr = T(lb_w(q)) * rho;
        const T even = wr * (k + T(4.5) * cu * cu), odd = wr * T(3) * cu;
        const T fa = even + odd, fb = even - odd;
        if (active) {
            push.put(fout, P, q, a - omega * (a - fa), rho);
            push.put(fout, P, q + 1, b - omega * (b - fb), rho);
        }
    }
}

// PSM collision, Eq. (32)-(37), of a cell cut by the solid (B0, uk0) and, when the warp-uniform flag `two` is
// set, by the second one parked in s2 (B = 0 there for the lanes that have none).
// For a pair of opposite directions (q, qbar) with a = f_q, b = f_qbar, E / O the even / odd part of f^eq(rho, u)
// and Ek / Ok those of f^eq(rho, u_k), Eq. (34) reads
//     Omega^s_q    = (b - (E - O)) - (a - (Ek + Ok)) = D + X,      D = Ek - E,  X = (Ok + O) - (a - b)
//     Omega^s_qbar = (a - (E + O)) - (b - (Ek - Ok)) = D - X
// and the fluid collision a - f^eq_q = Pp + Mm, b - f^eq_qbar = Pp - Mm with Pp = (a + b)/2 - E, Mm = (a - b)/2 - O,
// so both outputs come from one even part U = sum_k B_k D_k - (1 - B_tot) w+ Pp and one odd part
// V = sum_k B_k X_k - (1 - B_tot) w- Mm (w+ = w- for BGK): f*_q = a + (U + V), f*_qbar = b + (U - V).
// D is formed as t_q rho [(k_k - k) + 4.5 (c.u_k - c.u)(c.u_k + c.u)]: no cancellation of the two equilibria.
template <typename I, bool TRT, bool FAST, bool ONE, typename T>
__device__ __forceinline__ void psm_collide_stream(const T* sf, T omega, T rho, T ux, T uy, T uz,
                                                   T B0, const T (&uk0)[3], bool two_, const T* s2,
                                                   const LbPush<I>& push, T* __restrict__ fout, const LbmDev& P, bool active)
{
    const bool two = !ONE && two_;                                                  // ONE: the caller knows that no lane has a second solid
    const T k0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    const T kk0 = T(1) - T(1.5) * (uk0[0] * uk0[0] + uk0[1] * uk0[1] + uk0[2] * uk0[2]);
    const T Bsum = B0 + (two ? s2[0] : T(0));
    const T keep = T(1) - (Bsum < T(1) ? Bsum : T(1));                              // 1 - B_tot, Eq. (37)
    const T komega = keep * omega;
    const T komega_m = TRT ? keep * (T)P.omega_minus : komega;
    const T dk0 = kk0 - k0;
    T B1 = T(0), dk1 = T(0);
    if (two) { B1 = s2[0]; dk1 = s2[PSM_BLOCK] - k0; }
    {   // rest population: its own opposite, Omega^s = feq(rho,u_k) - feq(rho,u)
        const T f0 = sf[0], wr = T(lb_w(0)) * rho, fe = wr * k0;
        T acc = B0 * (wr * dk0);
        if (two) acc += B1 * (wr * dk1);
        if (FAST || active) push.template put<T, FAST>(fout, P, 0, f0 + (acc - komega * (f0 - fe)), rho);
    }
#pragma unroll
    for (int q = 1; q < LEDDS_Q; q += 2) {
        const T a = sf[q * PSM_BLOCK], b = sf[(q + 1) * PSM_BLOCK];
        const T wr = T(lb_w(q)) * rho, wr3 = T(3) * wr;
        const T cu = lb_cdot(q, ux, uy, uz), cuk = lb_cdot(q, uk0[0], uk0[1], uk0[2]);
        const T s = a + b, d = a - b;
        const T E = wr * (k0 + T(4.5) * cu * cu), O = wr3 * cu;
        T U = B0 * (wr * (dk0 + T(4.5) * (cuk - cu) * (cuk + cu)));                // B D
        T V = B0 * (wr3 * (cuk + cu) - d);                                          // B X
        if (two) {
            const T cu1 = lb_cdot(q, s2[2 * PSM_BLOCK], s2[3 * PSM_BLOCK], s2[4 * PSM_BLOCK]);
            U += B1 * (wr * (dk1 + T(4.5) * (cu1 - cu) * (cu1 + cu)));
            V += B1 * (wr3 * (cu1 + cu) - d);
        }
        U -= komega * (T(0.5) * s - E);                                             // Eq. (33): (1 - B_tot) Omega, BGK / TRT even part
        V -= komega_m * (T(0.5) * d - O);                                           //                               odd part
        if (FAST || active) {
            push.template put<T, FAST>(fout, P, q, a + (U + V), rho);               // Eq. (32)
            push.template put<T, FAST>(fout, P, q + 1, b + (U - V), rho);
        }
    }
}
