/*
 * oracle/lbm.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow CPU statement (fp64) of the D3Q19 BGK collide-and-stream step of
 * arxiv 2512.04997 (LEDDS), written from PAPER.md only.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_2512_04997_b200/; only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.
 *
 * What it follows:
 *   moments        PAPER.md:200-202  Eq. (22a), (22b)
 *   collide/stream PAPER.md:206-216  Eq. (23)-(25)
 *   BGK            PAPER.md:222      Eq. (26), relaxation time Eq. (27)
 *   TRT            PAPER.md:236-246  Eq. (29)-(31)
 *   equilibrium    PAPER.md:230      Eq. (28), c_s^2 = 1/3 (reading G17)
 *   boundaries     PAPER.md:254      "standard and velocity-modified bounce-back"
 *                                    (reading G19: halfway, link-wise)
 * Lattice units: dx = dt = 1.  Layout f[q*N + (z*ny + y)*nx + x].
 * Direction numbering (reading G18, a free choice the paper leaves to "any
 * textbook"): 0 rest; 1..6 = +x,-x,+y,-y,+z,-z; 7..18 the face
 * diagonals, every direction followed by its opposite.
 *
 * The step is written as the paper states it: for every cell, moments, then
 * collision (24), then streaming (25) as a PUSH of every post-collision
 * population to the neighbour it travels to.  Two arrays, no in-place tricks.
 * OpenMP is used on the cell loop only: every (cell, direction) writes one
 * distinct location, so the result does not depend on the thread count.
 *
 * Pins (tests/test_oracle_lbm.py): Taylor-Green decay, exact mass
 * conservation, pure streaming is a permutation, uniform equilibrium is a
 * fixed point, Couette profile, lattice isotropy sums; TRT: equals BGK for
 * tau^- = tau^+, (tau^+ - 1/2)(tau^- - 1/2) = 3/16, decay rate set by tau^+ alone.
 */
#include <math.h>
#include <stddef.h>
#include <string.h>

#define Q 19

static const int CX[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
static const int CY[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
static const int CZ[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
static const int OPP[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};

static double weight(int i) { return i == 0 ? 1.0 / 3.0 : (i <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }

void orc_lbm_lattice(int *cx, int *cy, int *cz, int *opp, double *t)
{
    for (int i = 0; i < Q; ++i) { cx[i] = CX[i]; cy[i] = CY[i]; cz[i] = CZ[i]; opp[i] = OPP[i]; t[i] = weight(i); }
}

/* Eq. (28) with c_s^2 = 1/3: rho t_i [1 + 3 c.u + 4.5 (c.u)^2 - 1.5 u.u] */
double orc_feq(int i, double rho, double ux, double uy, double uz)
{
    double cu = CX[i] * ux + CY[i] * uy + CZ[i] * uz;
    double uu = ux * ux + uy * uy + uz * uz;
    return rho * weight(i) * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
}

/* populations set to the equilibrium of prescribed fields.
 * rho == NULL -> 1, u == NULL -> 0.  u is u[3][N] (component-major). */
void orc_lbm_equilibrium(int nx, int ny, int nz, const double *rho, const double *u, double *f)
{
    size_t N = (size_t)nx * ny * nz;
    for (size_t c = 0; c < N; ++c) {
        double r = rho ? rho[c] : 1.0;
        double ux = u ? u[c] : 0.0, uy = u ? u[N + c] : 0.0, uz = u ? u[2 * N + c] : 0.0;
        for (int i = 0; i < Q; ++i) f[(size_t)i * N + c] = orc_feq(i, r, ux, uy, uz);
    }
}

/* Eq. (22a), (22b) */
void orc_lbm_moments(int nx, int ny, int nz, const double *f, double *rho, double *u)
{
    size_t N = (size_t)nx * ny * nz;
    for (size_t c = 0; c < N; ++c) {
        double r = 0, jx = 0, jy = 0, jz = 0;
        for (int i = 0; i < Q; ++i) {
            double v = f[(size_t)i * N + c];
            r += v; jx += v * CX[i]; jy += v * CY[i]; jz += v * CZ[i];
        }
        rho[c] = r; u[c] = jx / r; u[N + c] = jy / r; u[2 * N + c] = jz / r;
    }
}

/* Streaming (25) of one post-collision population fs = f_i^*(r) with the
 * boundary rule of reading G19.  bc[a] = 0 periodic, 1 walls.  u_wall is
 * [axis][side][component] (18 doubles), side 0 = low wall, 1 = high wall.
 * A link that leaves the box through one or more walled axes is reflected
 * into the opposite direction of the SAME cell, minus 6 t_i rho (c_i . u_w)
 * summed over the crossed walls; otherwise it travels to r + c_i with
 * periodic wrap. */
void orc_stream_one(int nx, int ny, int nz, const int *bc, const double *u_wall,
                    int x, int y, int z, int i, double fs, double rho, double *f_out)
{
    size_t N = (size_t)nx * ny * nz;
    int n[3] = {nx, ny, nz}, r[3] = {x, y, z}, c[3] = {CX[i], CY[i], CZ[i]}, t[3];
    int bounced = 0;
    double cuw = 0.0;
    for (int a = 0; a < 3; ++a) {
        t[a] = r[a] + c[a];
        if (t[a] < 0 || t[a] >= n[a]) {
            if (bc[a]) {
                int side = t[a] < 0 ? 0 : 1;
                const double *uw = u_wall + (a * 2 + side) * 3;
                cuw += c[0] * uw[0] + c[1] * uw[1] + c[2] * uw[2];
                bounced = 1;
            } else {
                t[a] = t[a] < 0 ? t[a] + n[a] : t[a] - n[a];
            }
        }
    }
    if (bounced)
        f_out[(size_t)OPP[i] * N + ((size_t)z * ny + y) * nx + x] = fs - 6.0 * weight(i) * rho * cuw;
    else
        f_out[(size_t)i * N + ((size_t)t[2] * ny + t[1]) * nx + t[0]] = fs;
}

/* Eq. (31): dt/tau^- for the TRT model, given dt/tau^+ (the "magic" combination
 * (tau^+ - 1/2)(tau^- - 1/2) = 3/16). */
double orc_trt_omega_minus(double omega_plus) { return 8.0 * (2.0 - omega_plus) / (8.0 - omega_plus); }

/* Collision term Omega_i of one cell.  omega_minus < 0: BGK, Eq. (26).  Otherwise TRT, Eq. (29)-(30),
 * written out as printed: f^+- = 0.5 (f_i +- f_ibar), same for the equilibria. */
double orc_collision(int i, const double *f, double rho, double ux, double uy, double uz, double omega, double omega_minus)
{
    double fe = orc_feq(i, rho, ux, uy, uz);
    if (omega_minus < 0.0) return -omega * (f[i] - fe);
    double feo = orc_feq(OPP[i], rho, ux, uy, uz);
    double fp = 0.5 * (f[i] + f[OPP[i]]), fm = 0.5 * (f[i] - f[OPP[i]]);
    double ep = 0.5 * (fe + feo), em = 0.5 * (fe - feo);
    return -omega * (fp - ep) - omega_minus * (fm - em);
}

/* One collide-and-stream step, Eq. (22)-(28); omega = dt/tau (tau^+ for TRT), omega_minus < 0 selects BGK.
 * omega = 0 gives pure streaming (used by the permutation pin). */
void orc_lbm_step(int nx, int ny, int nz, double omega, double omega_minus, const int *bc, const double *u_wall,
                  const double *f_in, double *f_out)
{
    size_t N = (size_t)nx * ny * nz;
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                size_t c = ((size_t)z * ny + y) * nx + x;
                double f[Q], rho = 0, jx = 0, jy = 0, jz = 0;
                for (int i = 0; i < Q; ++i) {
                    f[i] = f_in[(size_t)i * N + c];
                    rho += f[i]; jx += f[i] * CX[i]; jy += f[i] * CY[i]; jz += f[i] * CZ[i];
                }
                double ux = jx / rho, uy = jy / rho, uz = jz / rho;
                for (int i = 0; i < Q; ++i) {
                    double fs = omega_minus < 0.0 ? f[i] - omega * (f[i] - orc_feq(i, rho, ux, uy, uz))
                                                  : f[i] + orc_collision(i, f, rho, ux, uy, uz, omega, omega_minus);
                    orc_stream_one(nx, ny, nz, bc, u_wall, x, y, z, i, fs, rho, f_out);
                }
            }
}

/* nsteps steps, ping-pong between f and tmp; result always ends in f. */
void orc_lbm_run(int nx, int ny, int nz, double omega, double omega_minus, const int *bc, const double *u_wall,
                 double *f, double *tmp, int nsteps)
{
    size_t N = (size_t)nx * ny * nz;
    double *a = f, *b = tmp;
    for (int s = 0; s < nsteps; ++s) {
        orc_lbm_step(nx, ny, nz, omega, omega_minus, bc, u_wall, a, b);
        double *sw = a; a = b; b = sw;
    }
    if (a != f) memcpy(f, a, sizeof(double) * Q * N);
}
