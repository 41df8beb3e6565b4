// Device code of the PSM coupling kernels (Eq. 32-42).  Included by coupled.cu.
#pragma once
#include "lbm_kernels.cuh"

#define PSM_BLOCK 128
#define PSM_EMPTY 0xffffffffu

// Layout of the caller-owned coupling scratch (ledds_cpl_workspace_bytes):
//   slots[N]            uint2 per fluid cell: the (<= 2, lowest) ids of the solids cutting it, PSM_EMPTY
//                       when free.  Written by cpl_raster_kernel, consumed and reset by lbm_psm_kernel,
//                       so it is all-empty between steps.
//   sol[n][10]          per solid, lattice units: x_k[3], R_k, v_k[3], w_k[3] (predictor values)
//   flags[n][S^3]       uint8: box entry holds a partial of this step (set by lbm_psm_kernel, reset by
//                       cpl_reduce_kernel)
//   list2[1 + cap]      uint32: number and linear indices of the cells cut by two solids (written by the
//                       raster kernel, worked through by lbm_psm2_kernel, count reset by cpl_reduce_kernel)
//   box[n][S^3][6]      double: sum of the (cell, solid) terms of Eq. (41)-(42) over one run of
//                       consecutive cells of a lattice row inside a warp, stored at the run's first cell;
//                       S = 2H+2 cells per axis around floor(x_k)
struct CplDev {
    int n;
    double rc, inv_2rc;        // Eq. (40) in lattice units
    double inv_dx, vscale, wscale, origin[3];
    double fscale, mscale;     // lattice -> DEM units for force / torque
    int H, S;                  // box half-width, box width
    const double* x; const double* vp; const double* wp; const double* radius;   // particle order, DEM units
    uint2* slots;
    double* sol;
    uint8_t* flags;
    double* box;
    uint32_t* list2;           // [0] = count, [1..] = linear indices of the cells cut by two solids
    uint32_t list2_cap;
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

__device__ __forceinline__ int cpl_floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

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

// PSM collision of one cell cut by NS (1 or 2) solids, Eq. (32)-(37).  Written pair by pair (q, opposite q)
// so that no per-direction array besides f itself is live.  A solid with B = 0 contributes nothing, so lanes
// of a warp that are not cut run the same code with B = 0.
template <int NS>
__device__ __forceinline__ void psm_collide(double (&f)[LEDDS_Q], double omega, double rho, double ux, double uy,
                                            double uz, const double (&B)[NS], const double (&uk)[NS][3])
{
    const double k0 = 1.0 - 1.5 * (ux * ux + uy * uy + uz * uz);
    double kk[NS];
    double Bsum = 0.0;
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        kk[s] = 1.0 - 1.5 * (uk[s][0] * uk[s][0] + uk[s][1] * uk[s][1] + uk[s][2] * uk[s][2]);
        Bsum += B[s];
    }
    const double keep = 1.0 - (Bsum < 1.0 ? Bsum : 1.0);                              // 1 - B_tot, Eq. (37)
    const double komega = keep * omega;
    {   // rest population: its own opposite, Omega^s = feq(rho,u_k) - feq(rho,u)
        const double wr = lb_w(0) * rho, fe = wr * k0;
        double acc = 0.0;
#pragma unroll
        for (int s = 0; s < NS; ++s) acc += B[s] * (wr * kk[s] - fe);
        f[0] = f[0] + (acc - komega * (f[0] - fe));
    }
#pragma unroll
    for (int q = 1; q < LEDDS_Q; q += 2) {
        const double wr = lb_w(q) * rho;
        const double cu = lb_cdot(q, ux, uy, uz);
        const double ev = wr * (k0 + 4.5 * cu * cu), od = wr * 3.0 * cu;
        const double nq = f[q] - (ev + od), no = f[q + 1] - (ev - od);                   // f - feq(rho,u), Eq. (28)
        double acc_q = 0.0, acc_o = 0.0;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const double cuk = lb_cdot(q, uk[s][0], uk[s][1], uk[s][2]);
            const double evk = wr * (kk[s] + 4.5 * cuk * cuk), odk = wr * 3.0 * cuk;
            acc_q += B[s] * (no - (f[q] - (evk + odk)));                                // B Omega^s, Eq. (34), direction q
            acc_o += B[s] * (nq - (f[q + 1] - (evk - odk)));                            //                      its opposite
        }
        f[q] = f[q] + (acc_q - komega * nq);                                            // Eq. (32)-(33)
        f[q + 1] = f[q + 1] + (acc_o - komega * no);
    }
}

// Collision of a cell of a warp in which some cell is cut by a solid.  id[s] = PSM_EMPTY: no solid s here
// (B = 0).  Outputs per solid the terms of Eq. (41)-(42) in lattice units (rec) and the index of this cell
// in the solid's box (ent, -1 when there is no solid s).
template <int NS>
__device__ __forceinline__ void psm_cell(const LbmDev& P, const CplDev& C, int x, int y, int z, double (&f)[LEDDS_Q],
                                         double rho, double ux, double uy, double uz, const uint32_t (&id)[2],
                                         double (&rec)[2][6], int (&ent)[2])
{
    double B[NS], uk[NS][3], d[NS][3];
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const bool has = id[s] != PSM_EMPTY;
        const uint32_t k = has ? id[s] : 0u;
        const double2* sp = reinterpret_cast<const double2*>(C.sol + (size_t)k * 10);
        const double2 a0 = __ldg(sp), a1 = __ldg(sp + 1), a2 = __ldg(sp + 2), a3 = __ldg(sp + 3), a4 = __ldg(sp + 4);
        const double xk[3] = {a0.x, a0.y, a1.x}, Rk = a1.y;
        const double vk[3] = {a2.x, a2.y, a3.x}, wk[3] = {a3.y, a4.x, a4.y};
        const int fk[3] = {(int)floor(xk[0]), (int)floor(xk[1]), (int)floor(xk[2])};
        const int di[3] = {cpl_offset(x, fk[0], P.nx, !P.bc[0]), cpl_offset(y, fk[1], P.ny, !P.bc[1]),
                           cpl_offset(z, fk[2], P.nz, !P.bc[2])};
#pragma unroll
        for (int a = 0; a < 3; ++a) d[s][a] = (double)(fk[a] + di[a]) - xk[a];        // r_j - r_k, nearest image
        ent[s] = has ? ((di[2] + C.H) * C.S + (di[1] + C.H)) * C.S + (di[0] + C.H) : -1;
        const double dsc = cpl_dsc(Rk, C.rc, cpl_dist(d[s]));
        double beta = dsc * C.inv_2rc;                                                // Eq. (39)-(40)
        beta = beta > 1.0 ? 1.0 : beta;
        beta = (has && beta > 0.0) ? beta : 0.0;
        B[s] = beta * (P.tau - 0.5) / ((1.0 - beta) + (P.tau - 0.5));                 // Eq. (36)
        uk[s][0] = vk[0] + (wk[1] * d[s][2] - wk[2] * d[s][1]);                       // Eq. (35)
        uk[s][1] = vk[1] + (wk[2] * d[s][0] - wk[0] * d[s][2]);
        uk[s][2] = vk[2] + (wk[0] * d[s][1] - wk[1] * d[s][0]);
    }
    // Eq. (41): -B_k sum_i Omega^s_{i,k} c_i.  The sum is rho (u_k - u) identically (sum_i c_i f_i = rho u,
    // sum_i c_i f_i^eq(rho, v) = rho v, c_opp = -c), so it is formed from the moments.
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const double Br = B[s] * rho;
        const double dF[3] = {Br * (ux - uk[s][0]), Br * (uy - uk[s][1]), Br * (uz - uk[s][2])};   // lattice units
        rec[s][0] = dF[0]; rec[s][1] = dF[1]; rec[s][2] = dF[2];
        rec[s][3] = d[s][1] * dF[2] - d[s][2] * dF[1];                                // Eq. (42)
        rec[s][4] = d[s][2] * dF[0] - d[s][0] * dF[2];
        rec[s][5] = d[s][0] * dF[1] - d[s][1] * dF[0];
    }
    psm_collide<NS>(f, P.omega, rho, ux, uy, uz, B, uk);
}

// Sum the records of each run of consecutive lanes that hold the same solid id (a solid cuts a lattice row
// in consecutive cells) with a fixed shuffle tree, and let the first lane of the run write the sum into the
// solid's box at its own cell.  All 32 lanes call this; id = PSM_EMPTY marks a lane without a record.
__device__ __forceinline__ void psm_run_reduce(const CplDev& C, uint32_t id, int ent, double (&v)[6])
{
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const uint32_t prev = __shfl_up_sync(full, id, 1);
    const unsigned starts = __ballot_sync(full, lane == 0 || prev != id);          // bit l: lane l begins a run
    const unsigned above = lane == 31 ? 0u : (starts >> (lane + 1));
    const int len = above ? __ffs(above) : 32 - lane;                               // lanes from here to the end of my run
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            const double t = __shfl_down_sync(full, v[c], o);
            if (o < len) v[c] += t;
        }
    }
    if (id != PSM_EMPTY && ((starts >> lane) & 1u)) {
        const size_t e = (size_t)id * (size_t)(C.S * C.S * C.S) + (size_t)ent;
        double2* out = reinterpret_cast<double2*>(C.box + e * 6);
        out[0] = make_double2(v[0], v[1]);
        out[1] = make_double2(v[2], v[3]);
        out[2] = make_double2(v[4], v[5]);
        C.flags[e] = 1;
    }
}
