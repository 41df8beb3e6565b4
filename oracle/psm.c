/*
 * oracle/psm.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain CPU statement (fp64) of the partially-saturated-cell (PSM) fluid-solid
 * coupling of PAPER.md (arxiv 2512.04997) section 2.4 on top of the BGK
 * collide-and-stream of oracle/lbm.c.  Shares nothing with the CUDA path.
 *
 *   PSM collision        PAPER.md:270-275  Eq. (32), (33) with Omega_i = BGK (configs, G20) or TRT (Eq. 30)
 *   solid operator       PAPER.md:281      Eq. (34), overbar restored (reading G21)
 *   solid velocity       PAPER.md:285      Eq. (35), sign/index reading G22
 *   weighting            PAPER.md:289-295  Eq. (36), (37); only B_tot truncated (G23)
 *   solid fraction       PAPER.md:307-310  Eq. (39), (40) distance-based; Eq. (38) subdivision
 *   force / torque       PAPER.md:320-322  Eq. (41), (42), pre-collision f (G26)
 *   n_s <= 2 per cell    PAPER.md:515      the two lowest ids with beta > 0 (G24)
 *
 * Everything is in lattice units (dx = dt = 1, so dx^3/dt = 1); lattice node
 * (x,y,z) sits at integer coordinates; the caller converts particle state.
 * The order is the paper's (section 3.2.3): solid fractions per cell (found by
 * visiting, for every particle in ascending id, the cells of its bounding
 * box), then collision-streaming with the PSM operator, then the per-particle
 * reduction of the cell forces (here: a plain loop over the particle's cells).
 *
 * Pins (tests/test_oracle_psm.py): no particle == lbm.c bit for bit; sum_i
 * Omega^s = 0 and sum_i Omega^s c_i = rho (u_k - u); B(0)=0, B(1)=1; momentum
 * budget of the fluid; co-moving sphere feels no force; torque sign on a
 * spinning sphere; sum of beta ~ sphere volume; a third solid in a cell is
 * dropped by id (the step equals the step without it, bit for bit).
 * "parity unpinned": the
 * choice between the two readings of Eq. (34) beyond those identities (G21),
 * the truncation rule (G23).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>

#define Q 19
#define PI 3.14159265358979323846

double orc_feq(int i, double rho, double ux, double uy, double uz);
void orc_lbm_lattice(int *cx, int *cy, int *cz, int *opp, double *t);
void orc_stream_one(int nx, int ny, int nz, const int *bc, const double *u_wall,
                    int x, int y, int z, int i, double fs, double rho, double *f_out);

static int cx[Q], cy[Q], cz[Q], opp[Q];
static double t[Q];
static void tables(void) { orc_lbm_lattice(cx, cy, cz, opp, t); }

/* Eq. (40): radius of the sphere of volume dx^3 */
double orc_psm_rc(void) { return cbrt(3.0 / (4.0 * PI)); }

/* Eq. (39)-(40) */
double orc_psm_beta(double Rk, double dist)
{
    double Rc = orc_psm_rc();
    double dsc = (Rk + Rc) - dist;
    if (dsc <= 0.0) return 0.0;
    if (dsc >= 2.0 * Rc) return 1.0;
    return dsc / (2.0 * Rc);
}

/* Eq. (38), subdivision method: fraction of the ns^3 points s_i = r_j + ((a + 1/2)/ns - 1/2) (a = 0..ns-1 per
 * axis, "spread evenly inside the cell") that lie inside the sphere.  d = r_j - r_k. */
double orc_psm_beta_subdiv(const double *d, double Rk, int ns)
{
    int count = 0;
    double R2 = Rk * Rk;
    for (int c = 0; c < ns; ++c) {
        double sz = d[2] + (((double)c + 0.5) / (double)ns - 0.5);
        for (int b = 0; b < ns; ++b) {
            double sy = d[1] + (((double)b + 0.5) / (double)ns - 0.5);
            for (int a = 0; a < ns; ++a) {
                double sx = d[0] + (((double)a + 0.5) / (double)ns - 0.5);
                if (sx * sx + sy * sy + sz * sz < R2) ++count;
            }
        }
    }
    return (double)count / (double)(ns * ns * ns);
}

/* solid fraction of the cell whose centre is at d = r_j - r_k: subdiv = 0 distance-based (Eq. 39-40),
 * subdiv = ns > 0 subdivision with ns points per direction (Eq. 38) */
static double beta_of(const double *d, double Rk, int subdiv)
{
    if (subdiv > 0) return orc_psm_beta_subdiv(d, Rk, subdiv);
    return orc_psm_beta(Rk, sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
}

/* how far from the sphere centre a cell centre can be and still have beta > 0 */
static double reach_of(double Rk, int subdiv) { return subdiv > 0 ? Rk + 0.8661 : Rk + orc_psm_rc(); }

/* Eq. (36) */
double orc_psm_B(double beta, double tau) { return beta * (tau - 0.5) / ((1.0 - beta) + (tau - 0.5)); }

/* r_j - r_k with the lattice-node image nearest to the sphere on periodic axes */
static void node_minus_centre(const int *n, const int *bc, const int *r, const double *xk, double *d)
{
    for (int a = 0; a < 3; ++a) {
        d[a] = (double)r[a] - xk[a];
        if (!bc[a]) {
            if (d[a] > 0.5 * n[a]) d[a] = (double)(r[a] - n[a]) - xk[a];
            else if (d[a] < -0.5 * n[a]) d[a] = (double)(r[a] + n[a]) - xk[a];
        }
    }
}

/* Per (cell, solid): B_k and the momentum exchange sum_i Omega^s_{i,k} c_i,
 * optionally adding B_k Omega^s_{i,k} to fs[].  f = pre-collision populations. */
static double solid_terms(const int *n, const int *bc, double tau, const int *r, const double *f,
                          double rho, const double *u, const double *xk, const double *vk, const double *wk,
                          double Rk, int subdiv, double *d, double *sumOc, double *fs)
{
    node_minus_centre(n, bc, r, xk, d);
    double beta = beta_of(d, Rk, subdiv);
    double B = orc_psm_B(beta, tau);
    /* Eq. (35): u_k = v_k + w_k x (r_j - r_k) */
    double uk[3] = {vk[0] + (wk[1] * d[2] - wk[2] * d[1]),
                    vk[1] + (wk[2] * d[0] - wk[0] * d[2]),
                    vk[2] + (wk[0] * d[1] - wk[1] * d[0])};
    sumOc[0] = sumOc[1] = sumOc[2] = 0.0;
    for (int i = 0; i < Q; ++i) {
        int o = opp[i];
        /* Eq. (34): [f_ibar - feq_ibar(rho,u)] - [f_i - feq_i(rho,u_k)] */
        double Os = (f[o] - orc_feq(o, rho, u[0], u[1], u[2])) - (f[i] - orc_feq(i, rho, uk[0], uk[1], uk[2]));
        sumOc[0] += Os * cx[i]; sumOc[1] += Os * cy[i]; sumOc[2] += Os * cz[i];
        if (fs) fs[i] += B * Os;
    }
    return B;
}

/* One coupled LBM step.  np spheres: centre xk[3np], velocity vk, angular
 * velocity wk, radius Rk, all in lattice units.  Outputs: f_out, and the
 * hydrodynamic force F[3np] and torque M[3np] on every sphere (lattice units).
 * slots is scratch of 2*N ints.  status |= 2 when a third solid was dropped. */
double orc_collision(int i, const double *f, double rho, double ux, double uy, double uz, double omega, double omega_minus);

/* omega_minus < 0: BGK; else the TRT model of Eq. (29)-(31) as Omega_i in Eq. (33) */
void orc_psm_step(int nx, int ny, int nz, double tau, double omega_minus, int subdiv, const int *bc, const double *u_wall,
                  int np, const double *xk, const double *vk, const double *wk, const double *Rk,
                  const double *f_in, double *f_out, double *F, double *M, int *slots, int *status)
{
    size_t N = (size_t)nx * ny * nz;
    int n[3] = {nx, ny, nz};
    double omega = 1.0 / tau;
    tables();
    for (size_t c = 0; c < 2 * N; ++c) slots[c] = -1;

    /* (1) which solids cut which cell: ascending id, so a full cell keeps the two lowest */
    for (int k = 0; k < np; ++k) {
        double reach = reach_of(Rk[k], subdiv);
        int lo[3], hi[3];
        for (int a = 0; a < 3; ++a) { lo[a] = (int)ceil(xk[3 * k + a] - reach); hi[a] = (int)floor(xk[3 * k + a] + reach); }
        for (int z = lo[2]; z <= hi[2]; ++z)
            for (int y = lo[1]; y <= hi[1]; ++y)
                for (int x = lo[0]; x <= hi[0]; ++x) {
                    int r[3] = {x, y, z}, ok = 1;
                    for (int a = 0; a < 3; ++a)
                        if (r[a] < 0 || r[a] >= n[a]) { if (bc[a]) ok = 0; else r[a] = ((r[a] % n[a]) + n[a]) % n[a]; }
                    if (!ok) continue;
                    double d[3];
                    node_minus_centre(n, bc, r, xk + 3 * k, d);
                    if (beta_of(d, Rk[k], subdiv) <= 0.0) continue;
                    size_t c = ((size_t)r[2] * ny + r[1]) * nx + r[0];
                    if (slots[2 * c] < 0) slots[2 * c] = k;
                    else if (slots[2 * c] == k) {}
                    else if (slots[2 * c + 1] < 0) slots[2 * c + 1] = k;
                    else if (slots[2 * c + 1] != k) *status |= 2;
                }
    }

    /* (2) collision with the PSM operator, Eq. (32)-(33), then streaming */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                size_t c = ((size_t)z * ny + y) * nx + x;
                int r[3] = {x, y, z};
                double f[Q], fs[Q], rho = 0, j[3] = {0, 0, 0};
                for (int i = 0; i < Q; ++i) {
                    f[i] = f_in[(size_t)i * N + c];
                    rho += f[i]; j[0] += f[i] * cx[i]; j[1] += f[i] * cy[i]; j[2] += f[i] * cz[i];
                }
                double u[3] = {j[0] / rho, j[1] / rho, j[2] / rho};
                double Bsum = 0.0, solid[Q];
                for (int i = 0; i < Q; ++i) solid[i] = 0.0;
                for (int s = 0; s < 2; ++s) {
                    int k = slots[2 * c + s];
                    if (k < 0) continue;
                    double d[3], soc[3];
                    Bsum += solid_terms(n, bc, tau, r, f, rho, u, xk + 3 * k, vk + 3 * k, wk + 3 * k, Rk[k], subdiv, d, soc, solid);
                }
                double Btot = Bsum < 1.0 ? Bsum : 1.0;                       /* Eq. (37) */
                for (int i = 0; i < Q; ++i) {
                    double bgk = omega_minus < 0.0 ? -omega * (f[i] - orc_feq(i, rho, u[0], u[1], u[2]))
                                                   : orc_collision(i, f, rho, u[0], u[1], u[2], omega, omega_minus);
                    fs[i] = f[i] + ((1.0 - Btot) * bgk + solid[i]);          /* Eq. (32)-(33) */
                    orc_stream_one(nx, ny, nz, bc, u_wall, x, y, z, i, fs[i], rho, f_out);
                }
            }

    /* (3) Eq. (41), (42): per-particle sums over the cells the solid occupies */
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < np; ++k) {
        double reach = reach_of(Rk[k], subdiv), Fk[3] = {0, 0, 0}, Mk[3] = {0, 0, 0};
        int lo[3], hi[3];
        for (int a = 0; a < 3; ++a) { lo[a] = (int)ceil(xk[3 * k + a] - reach); hi[a] = (int)floor(xk[3 * k + a] + reach); }
        for (int z = lo[2]; z <= hi[2]; ++z)
            for (int y = lo[1]; y <= hi[1]; ++y)
                for (int x = lo[0]; x <= hi[0]; ++x) {
                    int r[3] = {x, y, z}, ok = 1;
                    for (int a = 0; a < 3; ++a)
                        if (r[a] < 0 || r[a] >= n[a]) { if (bc[a]) ok = 0; else r[a] = ((r[a] % n[a]) + n[a]) % n[a]; }
                    if (!ok) continue;
                    size_t c = ((size_t)r[2] * ny + r[1]) * nx + r[0];
                    if (slots[2 * c] != k && slots[2 * c + 1] != k) continue;
                    double f[Q], rho = 0, j[3] = {0, 0, 0};
                    for (int i = 0; i < Q; ++i) {
                        f[i] = f_in[(size_t)i * N + c];
                        rho += f[i]; j[0] += f[i] * cx[i]; j[1] += f[i] * cy[i]; j[2] += f[i] * cz[i];
                    }
                    double u[3] = {j[0] / rho, j[1] / rho, j[2] / rho}, d[3], soc[3];
                    double B = solid_terms(n, bc, tau, r, f, rho, u, xk + 3 * k, vk + 3 * k, wk + 3 * k, Rk[k], subdiv, d, soc, NULL);
                    double dF[3] = {-B * soc[0], -B * soc[1], -B * soc[2]};  /* Eq. (41) */
                    Fk[0] += dF[0]; Fk[1] += dF[1]; Fk[2] += dF[2];
                    Mk[0] += d[1] * dF[2] - d[2] * dF[1];                     /* Eq. (42) */
                    Mk[1] += d[2] * dF[0] - d[0] * dF[2];
                    Mk[2] += d[0] * dF[1] - d[1] * dF[0];
                }
        for (int a = 0; a < 3; ++a) { F[3 * k + a] = Fk[a]; M[3 * k + a] = Mk[a]; }
    }
}

/* per-cell total solid fraction sum_k beta_k (diagnostic for the volume pin) */
double orc_psm_beta_sum(int nx, int ny, int nz, const int *bc, const double *xk, double Rk, int subdiv)
{
    int n[3] = {nx, ny, nz};
    double s = 0.0;
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                int r[3] = {x, y, z};
                double d[3];
                node_minus_centre(n, bc, r, xk, d);
                s += beta_of(d, Rk, subdiv);
            }
    return s;
}
