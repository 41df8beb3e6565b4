/*
 * oracle/dem.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain CPU statement (fp64) of one DEM step for spheres as PAPER.md
 * (arxiv 2512.04997) defines it, in the paper's order and notation.  Shares
 * nothing with the CUDA path; only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.
 *
 *   contact test        PAPER.md:67-69, 96-100   Eq. (2), (6)  (strict, G7)
 *   normal              PAPER.md:102             Eq. (7)
 *   normal force        PAPER.md:116             Eq. (10) with the sign reading G1
 *   relative velocity   PAPER.md:120-124         Eq. (11), (12) (subscripts: G2)
 *   tangential history  PAPER.md:126-130         Eq. (13); previous value found by
 *                                                binary search in last step's sorted
 *                                                pair list
 *   spring-dashpot      PAPER.md:80              Eq. (4); Coulomb cap Eq. (5) (G8)
 *   torque              PAPER.md:138-140         Eq. (15), M/R shared by the pair
 *   walls               PAPER.md:142             static particle of infinite extent
 *                                                with a surface velocity (G13)
 *   damping             PAPER.md:982-1001        beta of (A.5), m* of (A.9); linear
 *                                                spring reading G5
 *   Hertz-Mindlin       PAPER.md:968-1001        (A.1)-(A.8), model = 1
 *   integration         PAPER.md:158-167, 188    Eq. (18a-c), (19d), (21a) (G11)
 *   pair list           PAPER.md:447-453, 492    unique pairs i<j sorted
 *                                                lexicographically
 *   uniform grid        PAPER.md:49, 431         spacing >= largest diameter
 *
 * A wall is partner id n + 2*axis + side (side 0 = low, 1 = high), so wall
 * contacts sort after all particle partners of the same i.
 *
 * Pins (tests/test_oracle_dem.py): restitution closed form, elastic energy
 * and momentum conservation, Psi_out = Psi_in - 7 mu (Eq. 51), free fall,
 * static rest on the floor, Newton's third law, cell-walk pair list ==
 * O(N^2) pair list; walls: restitution = eps_w (linear and Hertz, pins
 * m* = m_i and the wall's own zeta), elastic wall impact depth and duration
 * (linear: k_n,w; Hertz: R* = R_i and Y* from the wall's material).
 * "parity unpinned": gamma_t (G5), the projection of delta_t (G9), the
 * choice of predictor (G11).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int n;
    double lo[3], hi[3];
    int bc[3];               /* 0 periodic, 1 planar walls at lo/hi */
    double v_wall[18];       /* [axis][side][component] */
    double cell;             /* requested grid spacing */
    double dt, g[3], density;
    double kn, kt, restitution, mu;
    double kn_w, kt_w, restitution_w, mu_w;
    int model;               /* 0 linear spring-dashpot (configs, G4); 1 Hertz-Mindlin coefficients (A.1)-(A.8) */
    double young, poisson, young_w, poisson_w;   /* material of the spheres / of the walls */
} orc_dem_params;

#define PI 3.14159265358979323846

/* zeta = -beta of (A.5); e = exp(-pi zeta / sqrt(1 - zeta^2)) */
double orc_dem_zeta(double eps)
{
    if (eps >= 1.0) return 0.0;
    double l = log(eps);
    return -l / sqrt(l * l + PI * PI);
}

double orc_dem_mass(const orc_dem_params *p, double R) { return p->density * (4.0 / 3.0) * PI * R * R * R; }

/* uniform grid, SURVEY (c.2) step 2 / reading G14 */
void orc_dem_grid(const orc_dem_params *p, int *nc, double *inv_h)
{
    for (int a = 0; a < 3; ++a) {
        double L = p->hi[a] - p->lo[a];
        int n = (int)floor(L / p->cell);
        if (n < 1) n = 1;
        nc[a] = n;
        inv_h[a] = (double)n / L;
    }
}

static int cell_coord(const orc_dem_params *p, const int *nc, const double *inv_h, double x, int a)
{
    int c = (int)floor((x - p->lo[a]) * inv_h[a]);
    if (c < 0) c = 0;
    if (c > nc[a] - 1) c = nc[a] - 1;
    return c;
}

void orc_dem_keys(const orc_dem_params *p, const double *x, uint32_t *key)
{
    int nc[3]; double ih[3];
    orc_dem_grid(p, nc, ih);
    for (int i = 0; i < p->n; ++i) {
        int cx = cell_coord(p, nc, ih, x[3 * i], 0), cy = cell_coord(p, nc, ih, x[3 * i + 1], 1),
            cz = cell_coord(p, nc, ih, x[3 * i + 2], 2);
        key[i] = (uint32_t)(cx + nc[0] * (cy + nc[1] * cz));
    }
}

static int cmp_u64(const void *a, const void *b)
{
    uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/* stable order of particle ids by key (ties by ascending id, reading G15):
 * sort the unique 64-bit words key*2^32 + id. */
void orc_dem_order(int n, const uint32_t *key, uint32_t *idx)
{
    uint64_t *w = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(n > 0 ? n : 1));
    for (int i = 0; i < n; ++i) w[i] = ((uint64_t)key[i] << 32) | (uint32_t)i;
    qsort(w, (size_t)n, sizeof(uint64_t), cmp_u64);
    for (int i = 0; i < n; ++i) idx[i] = (uint32_t)(w[i] & 0xffffffffu);
    free(w);
}

/* r_i - r_j with the nearest image on periodic axes */
static void min_image(const orc_dem_params *p, const double *xi, const double *xj, double *d)
{
    for (int a = 0; a < 3; ++a) {
        d[a] = xi[a] - xj[a];
        if (!p->bc[a]) {
            double L = p->hi[a] - p->lo[a];
            if (d[a] > 0.5 * L) d[a] -= L;
            else if (d[a] < -0.5 * L) d[a] += L;
        }
    }
}

/* Eq. (6): delta_n = R_i + R_j - |r_i - r_j| */
static double overlap(const orc_dem_params *p, const double *x, const double *R, int i, int j)
{
    double d[3];
    min_image(p, x + 3 * i, x + 3 * j, d);
    return (R[i] + R[j]) - sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
}

static double wall_overlap(const orc_dem_params *p, const double *x, const double *R, int i, int w)
{
    int a = w >> 1, side = w & 1;
    double dist = side ? p->hi[a] - x[3 * i + a] : x[3 * i + a] - p->lo[a];
    return R[i] - dist;
}

static int emit_walls(const orc_dem_params *p, const double *x, const double *R, int i, uint32_t *pairs, int np, int cap)
{
    for (int w = 0; w < 6; ++w)
        if (p->bc[w >> 1] && wall_overlap(p, x, R, i, w) > 0.0) {
            if (np < cap) { pairs[2 * np] = (uint32_t)i; pairs[2 * np + 1] = (uint32_t)(p->n + w); }
            ++np;
        }
    return np;
}

/* O(N^2) definition of the pair list: all i<j with delta_n > 0, then the walls
 * of i.  Returns the count (may exceed cap; only cap pairs are stored). */
int orc_dem_pairs_brute(const orc_dem_params *p, const double *x, const double *R, uint32_t *pairs, int cap)
{
    int np = 0;
    for (int i = 0; i < p->n; ++i) {
        for (int j = i + 1; j < p->n; ++j)
            if (overlap(p, x, R, i, j) > 0.0) {
                if (np < cap) { pairs[2 * np] = (uint32_t)i; pairs[2 * np + 1] = (uint32_t)j; }
                ++np;
            }
        np = emit_walls(p, x, R, i, pairs, np, cap);
    }
    return np;
}

static int cmp_pair(const void *a, const void *b)
{
    const uint32_t *x = (const uint32_t *)a, *y = (const uint32_t *)b;
    if (x[0] != y[0]) return x[0] < y[0] ? -1 : 1;
    if (x[1] != y[1]) return x[1] < y[1] ? -1 : 1;
    return 0;
}

/* The same list through the uniform grid: for every particle walk the (up to)
 * 27 cells around its own, keep j > i with delta_n > 0, then sort
 * lexicographically.  idx/key = output of orc_dem_order. */
int orc_dem_pairs_cells(const orc_dem_params *p, const double *x, const double *R,
                        const uint32_t *key, const uint32_t *idx, uint32_t *pairs, int cap)
{
    int nc[3]; double ih[3];
    orc_dem_grid(p, nc, ih);
    size_t ncell = (size_t)nc[0] * nc[1] * nc[2];
    int *start = (int *)malloc(sizeof(int) * (ncell + 1));
    for (size_t c = 0; c <= ncell; ++c) start[c] = 0;
    for (int s = 0; s < p->n; ++s) start[key[idx[s]] + 1]++;
    for (size_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
    int np = 0;
    for (int i = 0; i < p->n; ++i) {
        int c[3] = {(int)(key[i] % nc[0]), (int)((key[i] / nc[0]) % nc[1]), (int)(key[i] / ((uint32_t)nc[0] * nc[1]))};
        int seen[27], nseen = 0;
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int q[3] = {c[0] + dx, c[1] + dy, c[2] + dz}, ok = 1;
                    for (int a = 0; a < 3; ++a) {
                        if (q[a] < 0 || q[a] >= nc[a]) {
                            if (p->bc[a]) ok = 0;
                            else q[a] = (q[a] + nc[a]) % nc[a];
                        }
                    }
                    if (!ok) continue;
                    int cell = q[0] + nc[0] * (q[1] + nc[1] * q[2]), dup = 0;
                    for (int k = 0; k < nseen; ++k) dup |= (seen[k] == cell);   /* tiny periodic grids */
                    if (dup) continue;
                    seen[nseen++] = cell;
                    for (int s = start[cell]; s < start[cell + 1]; ++s) {
                        int j = (int)idx[s];
                        if (j > i && overlap(p, x, R, i, j) > 0.0) {
                            if (np < cap) { pairs[2 * np] = (uint32_t)i; pairs[2 * np + 1] = (uint32_t)j; }
                            ++np;
                        }
                    }
                }
        np = emit_walls(p, x, R, i, pairs, np, cap);
    }
    free(start);
    qsort(pairs, (size_t)(np < cap ? np : cap), 2 * sizeof(uint32_t), cmp_pair);
    return np;
}

/* binary search of (i,j) in a lexicographically sorted pair list */
static int find_pair(const uint32_t *pairs, int np, uint32_t i, uint32_t j)
{
    int lo = 0, hi = np - 1;
    while (lo <= hi) {
        int mid = lo + (hi - lo) / 2;
        const uint32_t *q = pairs + 2 * mid;
        if (q[0] == i && q[1] == j) return mid;
        if (q[0] < i || (q[0] == i && q[1] < j)) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

static void cross(const double *a, const double *b, double *c)
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

/* Force and torque of every contact of the sorted pair list, Eq. (4)-(15),
 * reduced per particle, Eq. (1).  v, w are the velocities the force law sees
 * (the predictor values, reading G11).  dt_hist is the time increment of
 * Eq. (13) (0 when evaluating the forces of the initial state).
 * prev_* is last step's sorted pair list with its delta_t (np_prev pairs);
 * new_dt receives delta_t of every current pair.  status |= 4 for coincident
 * centres (pair skipped).  F, M are overwritten. */
void orc_dem_forces(const orc_dem_params *p, const double *x, const double *v, const double *w, const double *R,
                    int np, const uint32_t *pairs, int np_prev, const uint32_t *prev_pairs, const double *prev_dt,
                    double dt_hist, double *new_dt, double *F, double *M, int *status)
{
    int n = p->n;
    for (int k = 0; k < 3 * n; ++k) { F[k] = 0.0; M[k] = 0.0; }
    double zeta = orc_dem_zeta(p->restitution), zeta_w = orc_dem_zeta(p->restitution_w);
    for (int c = 0; c < np; ++c) {
        int i = (int)pairs[2 * c], j = (int)pairs[2 * c + 1];
        int wall = j >= n;
        double en[3], dn, Ri = R[i], Rj, mi = orc_dem_mass(p, Ri), mstar, vj[3], wj[3] = {0, 0, 0};
        double kn, kt, z, mu;
        if (!wall) {
            double d[3];
            min_image(p, x + 3 * i, x + 3 * j, d);
            double dist = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            dn = (Ri + R[j]) - dist;                               /* Eq. (6) */
            if (dist == 0.0) { *status |= 4; new_dt[3 * c] = new_dt[3 * c + 1] = new_dt[3 * c + 2] = 0.0; continue; }
            for (int a = 0; a < 3; ++a) en[a] = d[a] / dist;       /* Eq. (7) */
            Rj = R[j];
            double mj = orc_dem_mass(p, Rj);
            mstar = mi * mj / (mi + mj);                           /* (A.9) */
            for (int a = 0; a < 3; ++a) { vj[a] = v[3 * j + a]; wj[a] = w[3 * j + a]; }
            kn = p->kn; kt = p->kt; z = zeta; mu = p->mu;
        } else {
            int wl = j - n, ax = wl >> 1, side = wl & 1;
            dn = wall_overlap(p, x, R, i, wl);
            en[0] = en[1] = en[2] = 0.0;
            en[ax] = side ? -1.0 : 1.0;                            /* from the wall into the box */
            Rj = 0.0;                                              /* wall surface does not rotate */
            mstar = mi;                                            /* m_j = infinity */
            for (int a = 0; a < 3; ++a) vj[a] = p->v_wall[wl * 3 + a];
            kn = p->kn_w; kt = p->kt_w; z = zeta_w; mu = p->mu_w;
        }
        double gn, gt;
        if (p->model == 1) {
            /* Hertz-Mindlin coefficients of the pair.  (A.6) Y*, (A.7) G*, (A.8) R* (a wall is
             * a sphere of infinite radius: R* = R_i), (A.1) k_n, k_t, (A.3)-(A.4) S_n, S_t, (A.2) gamma with
             * beta of (A.5) = -zeta. */
            double Ei = p->young, ni = p->poisson, Ej = wall ? p->young_w : p->young, nj = wall ? p->poisson_w : p->poisson;
            double Ystar = 1.0 / ((1.0 - ni * ni) / Ei + (1.0 - nj * nj) / Ej);
            double Gstar = 1.0 / (2.0 * (2.0 - ni) * (1.0 + ni) / Ei + 2.0 * (2.0 - nj) * (1.0 + nj) / Ej);
            double Rstar = wall ? Ri : Ri * Rj / (Ri + Rj);
            double sq = sqrt(Rstar * dn);
            kn = (4.0 / 3.0) * Ystar * sq;
            kt = 8.0 * Gstar * sq;
            double Sn = 2.0 * Ystar * sq, St = 8.0 * Gstar * sq;
            gn = 2.0 * sqrt(5.0 / 6.0) * z * sqrt(Sn * mstar);
            gt = 2.0 * sqrt(5.0 / 6.0) * z * sqrt(St * mstar);
        } else {
            gn = 2.0 * z * sqrt(kn * mstar); gt = 2.0 * z * sqrt(kt * mstar);     /* reading G5 */
        }
        /* Eq. (11): v_rel = (v_i - v_j) - (R_i w_i + R_j w_j) x e_n */
        double rw[3], rwxe[3], vrel[3];
        for (int a = 0; a < 3; ++a) rw[a] = Ri * w[3 * i + a] + Rj * wj[a];
        cross(rw, en, rwxe);
        for (int a = 0; a < 3; ++a) vrel[a] = (v[3 * i + a] - vj[a]) - rwxe[a];
        double vn = vrel[0] * en[0] + vrel[1] * en[1] + vrel[2] * en[2];
        double vt[3];
        for (int a = 0; a < 3; ++a) vt[a] = vrel[a] - vn * en[a];                 /* Eq. (12) */
        double fn = kn * dn - gn * vn;                                            /* Eq. (10), G1, G6 */
        /* Eq. (13) with the history of the same pair, if it existed last step */
        double dt3[3] = {0, 0, 0};
        int h = find_pair(prev_pairs, np_prev, (uint32_t)i, (uint32_t)j);
        if (h >= 0) for (int a = 0; a < 3; ++a) dt3[a] = prev_dt[3 * h + a];
        double dte = dt3[0] * en[0] + dt3[1] * en[1] + dt3[2] * en[2];            /* G9 */
        for (int a = 0; a < 3; ++a) dt3[a] = (dt3[a] - dte * en[a]) + dt_hist * vt[a];
        double Ft[3];
        for (int a = 0; a < 3; ++a) Ft[a] = -kt * dt3[a] - gt * vt[a];            /* Eq. (4) */
        double ft = sqrt(Ft[0] * Ft[0] + Ft[1] * Ft[1] + Ft[2] * Ft[2]), fmax = mu * fabs(fn);
        if (ft > fmax) {                                                          /* Eq. (5), G8 */
            double s = fmax / ft;
            for (int a = 0; a < 3; ++a) { Ft[a] *= s; dt3[a] = -(Ft[a] + gt * vt[a]) / kt; }
        }
        for (int a = 0; a < 3; ++a) new_dt[3 * c + a] = dt3[a];
        double T[3];
        cross(en, Ft, T);                                                         /* Eq. (15): M/R = -e_n x F_t */
        for (int a = 0; a < 3; ++a) {
            double Fa = fn * en[a] + Ft[a];
            F[3 * i + a] += Fa;
            M[3 * i + a] += Ri * (-T[a]);
            if (!wall) { F[3 * j + a] -= Fa; M[3 * j + a] += Rj * (-T[a]); }
        }
    }
}

/* Eq. (18a) + the predictor of reading G11; periodic wrap into [lo, hi). */
void orc_dem_advance(const orc_dem_params *p, double *x, const double *v, const double *w,
                     const double *a, const double *alpha, double *vp, double *wp)
{
    double dt = p->dt;
    for (int i = 0; i < p->n; ++i)
        for (int k = 0; k < 3; ++k) {
            int q = 3 * i + k;
            double xn = x[q] + dt * v[q] + (0.5 * dt * dt) * a[q];
            if (!p->bc[k]) {
                double L = p->hi[k] - p->lo[k];
                if (xn >= p->hi[k]) xn -= L;
                else if (xn < p->lo[k]) xn += L;
            }
            x[q] = xn;
            vp[q] = v[q] + (0.5 * dt) * a[q];
            wp[q] = w[q] + (0.5 * dt) * alpha[q];
        }
}

/* Eq. (18b), (18c), (19c) for a sphere (alpha = M / I, I = 2/5 m R^2, Eq. 21a), (19d).
 * f_ext / m_ext (may be NULL) are extra per-particle force / torque. */
void orc_dem_kick(const orc_dem_params *p, const double *R, const double *F, const double *M,
                  const double *f_ext, const double *m_ext, double *v, double *w, double *a, double *alpha)
{
    double dt = p->dt;
    for (int i = 0; i < p->n; ++i) {
        double m = orc_dem_mass(p, R[i]), I = 0.4 * m * R[i] * R[i];
        for (int k = 0; k < 3; ++k) {
            int q = 3 * i + k;
            double Fq = F[q] + (f_ext ? f_ext[q] : 0.0), Mq = M[q] + (m_ext ? m_ext[q] : 0.0);
            double an = Fq / m + p->g[k], aln = Mq / I;
            v[q] = v[q] + (0.5 * dt) * (a[q] + an);
            w[q] = w[q] + (0.5 * dt) * (alpha[q] + aln);
            a[q] = an; alpha[q] = aln;
        }
    }
}
