// Device code of the PSM coupling kernels (Eq. 32-42).  Included by coupled.cu.
#pragma once
#include "lbm_kernels.cuh"

#define PSM_BLOCK 128
#define PSM_EMPTY 0xffffffffu

// Layout of the caller-owned coupling scratch (ledds_cpl_workspace_bytes):
//   slots[N]                      uint2 per fluid cell: the (<= 2, lowest) ids of the solids cutting it,
//                                 PSM_EMPTY when free.  Written by cpl_raster_kernel, consumed and reset
//                                 by lbm_psm_kernel, so it is all-empty between steps.
//   stamps[n][S][S][nseg]         uint32: LBM step that wrote the row partial
//   rows  [n][S][S][nseg][6]      double: sum over one lattice row segment of the (cell, solid) terms of
//                                 Eq. (41)-(42); S = 2H+2 rows per axis around floor(x_k)
struct CplDev {
    int n;
    double rc;                 // Eq. (40) in lattice units
    double inv_dx, vscale, wscale, origin[3];
    double fscale, mscale;     // lattice -> DEM units for force / torque
    int H, S, nseg, nbx;       // box half-width, box width, row segments per row, blocks along x
    uint32_t stamp;            // id of this LBM step (never 0)
    const double* x; const double* vp; const double* wp; const double* radius;   // particle order
    uint2* slots;
    uint32_t* stamps;
    double* rows;
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

// Ordinal of the PSM_BLOCK-wide block that holds unwrapped lattice coordinate p (periodic images
// of the row follow each other), used to number the row segments of one solid.
__device__ __forceinline__ int cpl_block_ordinal(int p, int nx, int nbx)
{
    const int per = cpl_floordiv(p, nx);
    return per * nbx + (p - per * nx) / PSM_BLOCK;
}

// lattice-unit position of solid k: x_k, floor(x_k), R_k
__device__ __forceinline__ void cpl_solid(const CplDev& C, uint32_t k, double* xk, int* fk, double& Rk)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        xk[a] = (C.x[3 * k + a] - C.origin[a]) * C.inv_dx;
        fk[a] = (int)floor(xk[a]);
    }
    Rk = C.radius[k] * C.inv_dx;
}

// PSM collision of one cell cut by one or two solids (B[1] = 0 when there is one), Eq. (32)-(37), and the
// momentum exchange sum_i Omega^s_{i,k} c_i of Eq. (41).  Written pair by pair (q, opposite q) so that no
// per-direction array besides f itself is live: the kernel keeps the register count of the plain one.
__device__ __forceinline__ void psm_collide(double (&f)[LEDDS_Q], double omega, double rho, double ux, double uy,
                                            double uz, const double (&B)[2], const double (&uk)[2][3],
                                            double (&soc)[2][3])
{
    const double k0 = 1.0 - 1.5 * (ux * ux + uy * uy + uz * uz);
    double kk[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        kk[s] = 1.0 - 1.5 * (uk[s][0] * uk[s][0] + uk[s][1] * uk[s][1] + uk[s][2] * uk[s][2]);
        soc[s][0] = soc[s][1] = soc[s][2] = 0.0;
    }
    const double Bsum = B[0] + B[1];
    const double keep = 1.0 - (Bsum < 1.0 ? Bsum : 1.0);                              // 1 - B_tot, Eq. (37)
    {   // rest population: its own opposite, Omega^s = feq(rho,u_k) - feq(rho,u)
        const double wr = lb_w(0) * rho, fe = wr * k0;
        double acc = 0.0;
#pragma unroll
        for (int s = 0; s < 2; ++s) acc += B[s] * ((f[0] - fe) - (f[0] - wr * kk[s]));
        f[0] = f[0] + (keep * (-omega * (f[0] - fe)) + acc);
    }
#pragma unroll
    for (int q = 1; q < LEDDS_Q; q += 2) {
        const double wr = lb_w(q) * rho;
        const double cu = lb_cdot(q, ux, uy, uz);
        const double ev = wr * (k0 + 4.5 * cu * cu), od = wr * 3.0 * cu;
        const double fe_q = ev + od, fe_o = ev - od;                                    // Eq. (28) for q and its opposite
        const double fq = f[q], fo = f[q + 1];
        double acc_q = 0.0, acc_o = 0.0;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const double cuk = lb_cdot(q, uk[s][0], uk[s][1], uk[s][2]);
            const double evk = wr * (kk[s] + 4.5 * cuk * cuk), odk = wr * 3.0 * cuk;
            const double Os_q = (fo - fe_o) - (fq - (evk + odk));                       // Eq. (34), direction q
            const double Os_o = (fq - fe_q) - (fo - (evk - odk));                       //           its opposite
            const double diff = Os_q - Os_o;                                            // c_q Os_q + c_o Os_o = c_q diff
            if (lb_cx(q) == 1) soc[s][0] += diff; else if (lb_cx(q) == -1) soc[s][0] -= diff;
            if (lb_cy(q) == 1) soc[s][1] += diff; else if (lb_cy(q) == -1) soc[s][1] -= diff;
            if (lb_cz(q) == 1) soc[s][2] += diff; else if (lb_cz(q) == -1) soc[s][2] -= diff;
            acc_q += B[s] * Os_q;
            acc_o += B[s] * Os_o;
        }
        f[q] = fq + (keep * (-omega * (fq - fe_q)) + acc_q);                            // Eq. (32)-(33)
        f[q + 1] = fo + (keep * (-omega * (fo - fe_o)) + acc_o);
    }
}

// What a cell contributes to one solid: force and torque terms of Eq. (41)-(42) in lattice units, and
// where the row partial they are summed into lives.
struct PsmRecord {
    double v[6];
    int row;        // (id * S + lz) * S + ly
    int xu;         // unwrapped x coordinate of this cell as seen from the solid (fk + di)
    int x0;         // unwrapped x coordinate of the first cell of the solid's box (fk - H)
};

// Collision of a cell cut by the solids id[0] (and id[1] unless PSM_EMPTY), Eq. (32)-(37), (39)-(40).
__device__ __forceinline__ void psm_cell(const LbmDev& P, const CplDev& C, const int* r, double (&f)[LEDDS_Q], double rho,
                                         double ux, double uy, double uz, const uint32_t (&id)[2], PsmRecord (&rec)[2])
{
    const int nl[3] = {P.nx, P.ny, P.nz};
    double B[2] = {0.0, 0.0}, uk[2][3] = {{0, 0, 0}, {0, 0, 0}}, d[2][3], soc[2][3];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (id[s] == PSM_EMPTY) continue;
        const uint32_t k = id[s];
        double xk[3], Rk;
        int fk[3], loc[3];
        cpl_solid(C, k, xk, fk, Rk);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int di = cpl_offset(r[a], fk[a], nl[a], !P.bc[a]);
            d[s][a] = (double)(fk[a] + di) - xk[a];                                   // r_j - r_k, nearest image
            loc[a] = di + C.H;
        }
        rec[s].row = ((int)k * C.S + loc[2]) * C.S + loc[1];
        rec[s].xu = fk[0] + loc[0] - C.H;
        rec[s].x0 = fk[0] - C.H;
        const double dsc = cpl_dsc(Rk, C.rc, cpl_dist(d[s]));
        const double beta = dsc >= 2.0 * C.rc ? 1.0 : (dsc > 0.0 ? dsc / (2.0 * C.rc) : 0.0);   // Eq. (39)
        B[s] = beta * (P.tau - 0.5) / ((1.0 - beta) + (P.tau - 0.5));                 // Eq. (36)
        const double vk[3] = {C.vp[3 * k] * C.vscale, C.vp[3 * k + 1] * C.vscale, C.vp[3 * k + 2] * C.vscale};
        const double wk[3] = {C.wp[3 * k] * C.wscale, C.wp[3 * k + 1] * C.wscale, C.wp[3 * k + 2] * C.wscale};
        uk[s][0] = vk[0] + (wk[1] * d[s][2] - wk[2] * d[s][1]);                       // Eq. (35)
        uk[s][1] = vk[1] + (wk[2] * d[s][0] - wk[0] * d[s][2]);
        uk[s][2] = vk[2] + (wk[0] * d[s][1] - wk[1] * d[s][0]);
    }
    psm_collide(f, P.omega, rho, ux, uy, uz, B, uk, soc);
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (id[s] == PSM_EMPTY) continue;
        const double dF[3] = {-B[s] * soc[s][0], -B[s] * soc[s][1], -B[s] * soc[s][2]};       // Eq. (41), lattice units
        rec[s].v[0] = dF[0]; rec[s].v[1] = dF[1]; rec[s].v[2] = dF[2];
        rec[s].v[3] = d[s][1] * dF[2] - d[s][2] * dF[1];                              // Eq. (42)
        rec[s].v[4] = d[s][2] * dF[0] - d[s][0] * dF[2];
        rec[s].v[5] = d[s][0] * dF[1] - d[s][1] * dF[0];
    }
}
