// Device code of the PSM stream-collide kernel (Eq. 32-42).  Included by coupled.cu.
#pragma once
#include "lbm_kernels.cuh"

#define PSM_BLOCK 128
#define PSM_MAXC 64

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

// A solid that may cut cells of the row segment a block works on (lattice units).
struct PsmCand { double xk[3], Rk; int fk[3]; uint32_t id, t; };

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

// lattice-unit state of the solid at sorted position t
__device__ __forceinline__ void psm_load_cand(const CplDev& C, uint32_t t, PsmCand& c)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        c.xk[a] = (C.xs[3 * t + a] - C.origin[a]) * C.inv_dx;
        c.fk[a] = (int)floor(c.xk[a]);
    }
    c.Rk = C.rs[t] * C.inv_dx;
    c.id = C.sidx[t];
    c.t = t;
}

// r_j - r_k (nearest image) and the index of cell r inside the solid's box of partials
__device__ __forceinline__ void psm_rel(const LbmDev& P, const CplDev& C, const int* r, const PsmCand& c, double* d, int* loc)
{
    const int nl[3] = {P.nx, P.ny, P.nz};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int di = cpl_offset(r[a], c.fk[a], nl[a], !P.bc[a]);
        d[a] = (double)(c.fk[a] + di) - c.xk[a];
        loc[a] = di + C.H;
    }
}

__device__ __forceinline__ double* psm_entry(const CplDev& C, uint32_t id, const int* loc)
{
    return C.boxes + ((((long long)id * C.S + loc[2]) * C.S + loc[1]) * C.S + loc[0]) * 6;
}

// keep the two lowest ids (G24); returns true when a solid had to be dropped
__device__ __forceinline__ bool psm_select(uint32_t id, int ci, uint32_t& id0, uint32_t& id1, int& c0, int& c1)
{
    if (id == id0 || id == id1) return false;
    if (id < id0) { const bool drop = id1 != 0xffffffffu; id1 = id0; c1 = c0; id0 = id; c0 = ci; return drop; }
    if (id < id1) { const bool drop = id1 != 0xffffffffu; id1 = id; c1 = ci; return drop; }
    return true;
}

// Collision of a cell cut by ns (1 or 2) solids + the partials of Eq. (41)-(42) into the solids' boxes.
__device__ __forceinline__ void psm_cell(const LbmDev& P, const CplDev& C, const int* r, double (&f)[LEDDS_Q], double rho,
                                         double ux, double uy, double uz, const PsmCand& p0, const PsmCand& p1, int ns)
{
    double B[2] = {0.0, 0.0}, uk[2][3] = {{0, 0, 0}, {0, 0, 0}}, d[2][3], soc[2][3];
    double* entry[2] = {nullptr, nullptr};
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (s >= ns) continue;
        const PsmCand& pc = s ? p1 : p0;
        int loc[3];
        psm_rel(P, C, r, pc, d[s], loc);
        const double dsc = cpl_dsc(pc.Rk, C.rc, cpl_dist(d[s]));
        const double beta = dsc >= 2.0 * C.rc ? 1.0 : dsc / (2.0 * C.rc);             // Eq. (39)
        B[s] = beta * (P.tau - 0.5) / ((1.0 - beta) + (P.tau - 0.5));                 // Eq. (36)
        const uint32_t t = pc.t;
        const double vk[3] = {C.vps[3 * t] * C.vscale, C.vps[3 * t + 1] * C.vscale, C.vps[3 * t + 2] * C.vscale};
        const double wk[3] = {C.wps[3 * t] * C.wscale, C.wps[3 * t + 1] * C.wscale, C.wps[3 * t + 2] * C.wscale};
        uk[s][0] = vk[0] + (wk[1] * d[s][2] - wk[2] * d[s][1]);                       // Eq. (35)
        uk[s][1] = vk[1] + (wk[2] * d[s][0] - wk[0] * d[s][2]);
        uk[s][2] = vk[2] + (wk[0] * d[s][1] - wk[1] * d[s][0]);
        entry[s] = psm_entry(C, pc.id, loc);
    }
    psm_collide(f, P.omega, rho, ux, uy, uz, B, uk, soc);
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (s >= ns) continue;
        const double dF[3] = {-B[s] * soc[s][0], -B[s] * soc[s][1], -B[s] * soc[s][2]};       // Eq. (41), lattice units
        double* e = entry[s];
        e[0] = dF[0]; e[1] = dF[1]; e[2] = dF[2];
        e[3] = d[s][1] * dF[2] - d[s][2] * dF[1];                                     // Eq. (42)
        e[4] = d[s][2] * dF[0] - d[s][0] * dF[2];
        e[5] = d[s][0] * dF[1] - d[s][1] * dF[0];
    }
}

// A dropped solid (more than two in a cell, PAPER.md:515 allows two) gets a zero partial so that its
// reduction never reads a stale entry.
__device__ __forceinline__ void psm_zero_dropped(const LbmDev& P, const CplDev& C, const int* r, const PsmCand& pc)
{
    double dd[3]; int loc[3];
    psm_rel(P, C, r, pc, dd, loc);
    if (!(cpl_dsc(pc.Rk, C.rc, cpl_dist(dd)) > 0.0)) return;
    double* e = psm_entry(C, pc.id, loc);
    for (int c = 0; c < 6; ++c) e[c] = 0.0;
}
