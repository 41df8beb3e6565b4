/*
 * ledds.h -- C ABI of libledds.so: the data-parallel hot path of one coupled
 * Lattice-Boltzmann / Discrete-Element time step of arxiv 2512.04997 (LEDDS),
 * hand-written CUDA for sm_100a, fp64 (optionally an fp32 lattice), one GPU.
 *
 * Conventions (all entry points)
 *   - Returns int: LEDDS_OK or a negative LEDDS_E* code.  Never throws, never aborts.
 *   - Every array argument is a DEVICE pointer owned by the caller unless it says "host".
 *     The library allocates NO device memory; sizes come from the *_workspace_bytes queries.
 *     Device pointers must be 16-byte aligned (LEDDS_EALIGN otherwise).
 *   - All work is ordered on the caller's stream (a cudaStream_t passed as void*; NULL = legacy
 *     default stream) and the call returns without synchronising.  ledds_coupled_step runs the
 *     contact pipeline of the DEM step beside the lattice kernels on an internal stream that is
 *     forked from and joined back into the caller's stream with events (capturable in a CUDA graph).
 *   - Handles (ledds_lbm, ledds_dem) are small HOST structs that hold parameters and step
 *     parity only; free them with *_destroy.
 *   - `status` is a caller-owned device int32[4]; word 0 collects asynchronous fault bits
 *     (LEDDS_ST_*), to be read by the caller after it synchronises.  Words 1..3 are scratch.
 *   - Particle arrays are in the caller's (unsorted) particle order; vectors are [n][3].
 *
 * Lattice (Eq. 22-28): D3Q19, c_s^2 = 1/3, dx = dt = 1.
 *   Direction numbering (fixed here; the paper leaves it to "any textbook"):
 *     q : 0      1   2   3   4   5   6    7    8    9    10   11   12   13   14   15   16   17   18
 *     cx: 0      1  -1   0   0   0   0    1   -1    1   -1    1   -1    1   -1    0    0    0    0
 *     cy: 0      0   0   1  -1   0   0    1   -1   -1    1    0    0    0    0    1   -1    1   -1
 *     cz: 0      0   0   0   0   1  -1    0    0    0    0    1   -1   -1    1    1   -1   -1    1
 *   opposite(q) = q odd ? q+1 : q-1 (q >= 1); weights 1/3 (q=0), 1/18 (1..6), 1/36 (7..18).
 *   Canonical population layout: f[q*N + (z*ny + y)*nx + x], N = nx*ny*nz, x fastest.
 *   Lattice node (x,y,z) sits at integer coordinates; a wall lies half a spacing outside the
 *   outermost nodes (halfway bounce-back).
 */
#ifndef LEDDS_H
#define LEDDS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LEDDS_OK 0
#define LEDDS_EINVAL (-1)     /* bad size / parameter / null pointer                     */
#define LEDDS_EALIGN (-2)     /* device pointer not 16-byte aligned                      */
#define LEDDS_ECAPACITY (-3)  /* a caller-provided buffer or capacity is too small       */
#define LEDDS_ECUDA (-4)      /* CUDA launch/runtime error (cudaGetLastError is kept)    */

#define LEDDS_ST_CONTACT_OVERFLOW 1 /* a particle had more than max_contacts contacts    */
#define LEDDS_ST_SOLID_OVERFLOW 2   /* a fluid cell was cut by more than 2 solids        */
#define LEDDS_ST_COINCIDENT 4       /* two sphere centres coincide (pair skipped)        */
#define LEDDS_ST_NONFINITE 8        /* a non-finite force was produced                   */
#define LEDDS_ST_RADIUS_RANGE 16    /* a radius is larger than the grids were sized for: 2 R > DEM cell width
                                       (contacts beyond the 27-cell walk are missed) or R > r_max of the
                                       coupling (the solid's cut cells are truncated)     */
#define LEDDS_ST_OUT_OF_BOX 32      /* a sphere centre lies outside a walled box (its cell index was clamped) */

typedef struct ledds_lbm ledds_lbm;
typedef struct ledds_dem ledds_dem;

/* ------------------------------------------------------------------------------------ LBM
 * Fused D3Q19 stream-collide (BGK or TRT), Eq. (22)-(31), boundaries PAPER.md:254. */
typedef struct {
    int nx, ny, nz;          /* lattice size, x fastest                                           */
    double tau;              /* relaxation time in units of dt, > 0.5 (Eq. 27)                    */
    int bc[3];               /* per axis: 0 periodic, 1 walls (halfway bounce-back) on both sides */
    double u_wall[3][2][3];  /* wall velocity [axis][side: 0 low, 1 high][component], lattice units;
                                velocity-modified bounce-back: f -= 6 t_i rho (c_i . u_wall)      */
    int layout;              /* must be 0: two-lattice streaming, f holds 2 x 19 x N doubles (PAPER.md:404:
                                "two populations").  No other layout exists; anything else: LEDDS_EINVAL */
    int variant;             /* index width of the kernel: 0 auto (32-bit when 19 N < 2^32, else 64-bit),
                                1 = 0, 3 forces the 64-bit path (tests).  Anything else: LEDDS_EINVAL     */
    int collision;           /* 0 = BGK, Eq. (26).  1 = TRT, Eq. (29)-(30) with tau^+ = tau and tau^- of
                                Eq. (31); also the Omega_i of the PSM collision Eq. (33)  */
} ledds_lbm_params;

/* f_bytes: size of the population buffer the caller must allocate for this layout. */
int ledds_lbm_workspace_bytes(const ledds_lbm_params* p, size_t* f_bytes);

/* Creates the handle and sets f to the equilibrium (Eq. 28) of rho[N] (NULL -> 1) and
 * u[3][N] component-major (NULL -> 0).  f: device, f_bytes large. */
int ledds_lbm_init(ledds_lbm** h, const ledds_lbm_params* p, double* f, const double* rho, const double* u,
                   void* stream);

/* Loads a canonical population field f_canonical[19*N] as the current state (parity tests). */
int ledds_lbm_import(ledds_lbm* h, double* f, const double* f_canonical, void* stream);

/* nsteps collide-and-stream steps (Eq. 23-26) in place in the caller's buffer. */
int ledds_lbm_step(ledds_lbm* h, double* f, int nsteps, void* stream);

/* Current state in canonical layout and/or its moments (Eq. 22); any output may be NULL.
 * f_canonical[19*N], rho[N], u[3][N]. */
int ledds_lbm_export(ledds_lbm* h, const double* f, double* f_canonical, double* rho, double* u, void* stream);

/* Pointer (inside f) of the current canonical 19*N field; host-side query, no device work. */
const double* ledds_lbm_current(const ledds_lbm* h, const double* f);

int ledds_lbm_destroy(ledds_lbm* h);

/* Single-precision variant of the plain LBM calls above (the paper runs most of its validations and one
 * of its two performance curves in fp32).  Same operation, layout (two lattices of
 * 19 x N floats), boundaries and collision models; all arithmetic in fp32; rho, u and f_canonical are float
 * arrays.  A handle made by
 * ledds_lbm_init_f32 is accepted by the _f32 calls and ledds_lbm_destroy only, a handle made by
 * ledds_lbm_init by the fp64 calls only (LEDDS_EINVAL otherwise).  ledds_coupled_step_f32 below takes the
 * fp32 handle. */
int ledds_lbm_workspace_bytes_f32(const ledds_lbm_params* p, size_t* f_bytes);
int ledds_lbm_init_f32(ledds_lbm** h, const ledds_lbm_params* p, float* f, const float* rho, const float* u,
                       void* stream);
int ledds_lbm_import_f32(ledds_lbm* h, float* f, const float* f_canonical, void* stream);
int ledds_lbm_step_f32(ledds_lbm* h, float* f, int nsteps, void* stream);
int ledds_lbm_export_f32(ledds_lbm* h, const float* f, float* f_canonical, float* rho, float* u, void* stream);

/* ------------------------------------------------------------------------------------ DEM
 * One DEM step for spheres, PAPER.md:63-142 (Eq. 1-15), 158-192 (Eq. 18-21), 431-511:
 *   drift (18a) + predictor -> cell keys on a uniform grid (spacing >= largest diameter,
 *   PAPER.md:49, 431) -> stable sort of particles by key -> cell ranges -> contact detection
 *   (Eq. 2, 6) by walking the 27 neighbour cells -> linear spring-dashpot normal/tangential
 *   force with Coulomb cap (Eq. 4-13), torque (Eq. 15), tangential history carried per contact
 *    -> per-particle sums (Eq. 1) without global atomics -> kick (18b-c, 19d).
 * Damping: gamma = 2 zeta sqrt(k m*), zeta = -ln e / sqrt(pi^2 + ln^2 e) (A.5), m* of (A.9).
 * A wall is a static infinite particle with a surface velocity; its partner id
 * is n + 2*axis + side. */
typedef struct {
    int n;                         /* particles, >= 0 (n = 0: every DEM call is a no-op and the
                                      array arguments may be NULL)                               */
    double lo[3], hi[3];           /* box                                                        */
    int bc[3];                     /* 0 periodic, 1 planar walls at lo/hi                        */
    double v_wall[3][2][3];        /* wall surface velocity [axis][side][component]              */
    double cell;                   /* requested grid spacing, >= 2 max radius; the grid has
                                      floor((hi-lo)/cell) cells per axis (>= 3 on periodic axes) */
    double dt, g[3], density;      /* step, gravity (already buoyancy-corrected, Eq. 56), rho_p  */
    double kn, kt, restitution, mu;          /* particle-particle spring-dashpot + Coulomb       */
    double kn_w, kt_w, restitution_w, mu_w;  /* particle-wall                                    */
    int max_contacts;              /* history slots per particle, 1..32 (walls included)         */
    int model;                     /* 0 = linear spring-dashpot with the k, restitution above;
                                      1 = Hertz-Mindlin coefficients per contact from the materials,
                                      PAPER.md:968-1001 (A.1)-(A.8); kn, kt are then ignored          */
    double young, poisson;         /* Young's modulus and Poisson ratio of the spheres (model 1)  */
    double young_w, poisson_w;     /* ... of the walls                                            */
    int sort_every_step;           /* 0: the radix passes of a step are skipped when the cell keys are still in
                                      order (the sort would be the identity; the result is the same);
                                      1: always run them (measurement)                             */
    int no_single_block;           /* 0: a system of up to 4 096 particles on a grid of up to 32 768 cells is
                                      stepped by ONE launch per step (a cluster of 8 thread blocks with cluster
                                      barriers between the phases) instead of twelve dependent launches; same
                                      results: the order and the lists are unique, the arithmetic is the same;
                                      1: always the chain of kernels (measurement, tests)          */
    int cell_order;                /* how the chain of kernels orders the particles by cell: 0 = counting sort over
                                      the cells when the grid has at most 4 n cells, radix passes over the keys
                                      otherwise; 1 = always the radix passes; 2 = always the counting sort.  The
                                      order (cell key, then id) is the same either way, bit for bit  */
} ledds_dem_params;

/* scratch and history are caller-owned but belong to the handle between calls: the library keeps the particle state
 * there in its own ("home") order while a call runs, and the last sort, the contact lists and the tangential history
 * between calls.  The caller's arrays x, v, w, a, alpha are read when a call begins and written when it ends; they may
 * be changed by the caller between calls (the next call picks the changes up), scratch and history may not. */
int ledds_dem_workspace_bytes(const ledds_dem_params* p, size_t* scratch_bytes, size_t* history_bytes);

/* Creates the handle, clears history/scratch, evaluates the contacts of the initial state with
 * delta_t = 0 and returns a(0) = F/m + g, alpha(0) = M/I (I = 2/5 m R^2, Eq. 21a).  x, v, w,
 * radius: in.  a, alpha: out. */
int ledds_dem_init(ledds_dem** h, const ledds_dem_params* p, const double* x, const double* v, const double* w,
                   const double* radius, double* a, double* alpha, void* history, void* scratch, int32_t* status,
                   void* stream);

/* nsteps DEM steps.  f_ext / m_ext: optional extra force / torque per particle ([n][3], may be NULL). */
int ledds_dem_step(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                   const double* f_ext, const double* m_ext, void* history, void* scratch, int32_t* status,
                   int nsteps, void* stream);

/* Results of the last force evaluation, for parity checks.  Any output may be NULL.
 *   sorted_idx[n]: particle ids ordered by (cell key, id);  sorted_key[n]: their keys;
 *   pairs[2*pair_cap]: canonical contact list, i < j, sorted lexicographically (walls as j >= n);
 *   n_pairs[1]: number of contacts (may exceed pair_cap: then only pair_cap are written);
 *   pair_dt[3*pair_cap]: delta_t of each listed contact, seen from i;
 *   force[3n], torque[3n]: contact force / torque per particle (Eq. 1), without gravity. */
int ledds_dem_query(ledds_dem* h, const void* history, const void* scratch, uint32_t* sorted_idx,
                    uint32_t* sorted_key, uint32_t* pairs, double* pair_dt, uint32_t pair_cap, uint32_t* n_pairs,
                    double* force, double* torque, void* stream);

int ledds_dem_destroy(ledds_dem* h);

/* The cell order of a particle set -- the linear cell index of every particle and the stable radix sort of the ids
 * by it, PAPER.md:388, 431-439 -- for callers that can neither allocate nor bring a scratch buffer (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  No handle, no workspace: the sort's scratch
 * is a static device array inside the library (about 4.4 MiB, held by every GPU that loads the library until the
 * process exits), so n is limited to LEDDS_CELL_ORDER_STATIC_MAX_N; a larger p->n returns LEDDS_ECAPACITY and
 * nothing is launched.  The call allocates no host or device memory and creates no stream or event.
 *   p: as for ledds_dem_init (validated in the same way); n, lo, hi, bc and cell decide the result;
 *   x[3n]: in, device, positions by particle id (a position outside the box takes the nearest cell, as in a step);
 *   sorted_idx[n], sorted_key[n]: out, device: particle ids ordered by (cell key, id) and their keys -- the same
 *   arrays ledds_dem_query returns after ledds_dem_init on these positions, bit for bit.
 * All calls on one device share the static array: calls that overlap on the GPU (different streams, or different
 * host threads without ordering between their streams) race and give undefined results; calls on one stream, or
 * ordered by events, are safe.  Works on the current device. */
#define LEDDS_CELL_ORDER_STATIC_MAX_N 262144
int ledds_dem_cell_order_static(const ledds_dem_params* p, const double* x, uint32_t* sorted_idx, uint32_t* sorted_key,
                                void* stream);
int ledds_dem_cell_order_static_max_n(void);   /* LEDDS_CELL_ORDER_STATIC_MAX_N of the loaded library */

/* Single-precision variant of the DEM calls (the paper runs most of its DEM validations in single precision and shows
 * fp32 next to fp64 energy curves, Appendix B).  Same pipeline and arguments on float
 * arrays; the particle state, the sorted records, the predictor velocities, the contact history and every operation
 * of the step are fp32.  Rules for the discrete decisions: the cell of a particle is floor((x - lo) * inv_h) in fp32
 * with inv_h = (float)(n_cells / L); a pair is in contact when (R_i + R_j) - sqrt(d.d) > 0 in fp32, d the fp32
 * difference of the fp32 positions (nearest image), summed as (dx dx + dy dy) + dz dz; a wall when R - distance > 0
 * in fp32.  Ordering (cell key, then id) and the canonical pair list are defined as for fp64, on those decisions.
 * A handle made by ledds_dem_init_f32 is accepted by the _f32 calls and ledds_dem_destroy only, and not by
 * ledds_coupled_step (LEDDS_EINVAL). */
int ledds_dem_workspace_bytes_f32(const ledds_dem_params* p, size_t* scratch_bytes, size_t* history_bytes);
int ledds_dem_init_f32(ledds_dem** h, const ledds_dem_params* p, const float* x, const float* v, const float* w,
                       const float* radius, float* a, float* alpha, void* history, void* scratch, int32_t* status,
                       void* stream);
int ledds_dem_step_f32(ledds_dem* h, float* x, float* v, float* w, float* a, float* alpha, const float* radius,
                       const float* f_ext, const float* m_ext, void* history, void* scratch, int32_t* status, int nsteps,
                       void* stream);
int ledds_dem_query_f32(ledds_dem* h, const void* history, const void* scratch, uint32_t* sorted_idx,
                        uint32_t* sorted_key, uint32_t* pairs, float* pair_dt, uint32_t pair_cap, uint32_t* n_pairs,
                        float* force, float* torque, void* stream);

/* -------------------------------------------------------------------------------- coupling
 * Partially saturated cells: solid fraction Eq. (39)-(40), weights Eq. (36)-(37),
 * PSM collision Eq. (32)-(35) fused into the stream-collide pass, hydrodynamic force and torque
 * Eq. (41)-(42) reduced per particle; order of the step PAPER.md:427, 515-532, sub-stepping
 * PAPER.md:258. */
typedef struct {
    int n_sub;            /* DEM sub-steps per LBM step; LBM dt = n_sub * dem.dt                  */
    int solid_fraction;   /* 0 = distance-based Eq. (39)-(40); 1 = subdivision Eq. (38), 10^3 points per
                             cell: + 8 B x (2H+2)^3 of scratch per solid             */
    double dx;            /* lattice spacing in DEM length units                                  */
    double rho_f;         /* fluid reference density in DEM units (lattice rho = 1)               */
    double origin[3];     /* DEM coordinates of lattice node (0,0,0)                              */
} ledds_cpl_params;

/* Size of the coupling scratch: one uint32 pair per fluid cell (the solids cutting it), 80 B per solid
 * (its state in lattice units) and 96 B per solid (fixed-point accumulators of Eq. (41)-(42)).
 * r_max = largest radius. */
int ledds_cpl_workspace_bytes(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c,
                              const double r_max, size_t* cpl_scratch_bytes);

/* Prepares cpl_scratch (all cell slots empty, accumulators at zero).  Call once before the first
 * ledds_coupled_step on this scratch, with the same lbm / dem / c / r_max. */
int ledds_cpl_init(const ledds_lbm* lbm, const ledds_dem* dem, const ledds_cpl_params* c, double r_max,
                   void* cpl_scratch, void* stream);

/* nsteps coupled steps.  f_hyd / m_hyd [n][3]: in = hydrodynamic force / torque of the previous
 * LBM step (zeros before the first), out = those of this step (DEM units).  The lattice and the DEM
 * box must have the same topology (bc); a periodic lattice axis must be at least 2 (2H+2) long
 * (unique nearest image), H = ceil(r_max/dx + 0.6204).  LEDDS_EINVAL otherwise.  f_hyd / m_hyd are exact
 * sums (2^-83 fixed point) of the per-cell terms, so they do not depend on the order of execution. */
int ledds_coupled_step(ledds_lbm* lbm, ledds_dem* dem, const ledds_cpl_params* c, double r_max, double* f,
                       double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                       double* f_hyd, double* m_hyd, void* history, void* scratch, void* cpl_scratch,
                       int32_t* status, int nsteps, void* stream);

/* The coupled step on an fp32 lattice (handle from ledds_lbm_init_f32, f = 2 x 19 x N floats): the populations,
 * their moments (Eq. 22) and the collision (Eq. 26 / 29-30, 32-37) are single precision; the geometry of the
 * solids (Eq. 35, 39-40, 38), the sums of Eq. (41)-(42) and the whole DEM step stay double, so the cells a
 * solid cuts, the contact list and the order-independence of f_hyd / m_hyd are those of the fp64 call.  All other
 * arguments, the scratch buffers (ledds_cpl_workspace_bytes / ledds_cpl_init take either kind of handle) and the
 * error behaviour are as for ledds_coupled_step; LEDDS_EINVAL when the handle's precision does not match. */
int ledds_coupled_step_f32(ledds_lbm* lbm, ledds_dem* dem, const ledds_cpl_params* c, double r_max, float* f,
                           double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                           double* f_hyd, double* m_hyd, void* history, void* scratch, void* cpl_scratch,
                           int32_t* status, int nsteps, void* stream);

/* ------------------------------------------------------------------------------ measurement
 * Optional per-kernel timing with CUDA events recorded on the launching stream around each kernel
 * group, and a count of the kernels this library has launched.  Host-side state, off by default. */
#define LEDDS_K_LBM 0          /* stream-collide (plain or PSM) */
#define LEDDS_K_DEM_KEYS 1     /* drift + predictor + cell keys */
#define LEDDS_K_DEM_SORT 2     /* histogram + radix passes      */
#define LEDDS_K_DEM_GATHER 3   /* sorted copies + cell ranges   */
#define LEDDS_K_DEM_CONTACT 4  /* contact detection + forces    */
#define LEDDS_K_DEM_KICK 5     /* velocity update               */
#define LEDDS_K_CPL_REDUCE 6   /* fixed point -> F_sf, M_sf      */
#define LEDDS_K_CPL_RASTER 7   /* solids -> per-cell slots      */
/* enable != 0: start recording (previous records are dropped); 0: stop and drop. */
int ledds_profile(int enable);
/* Sum of the recorded durations [ms] and number of recorded launches of one kernel group;
 * synchronises on the recorded events.  total_ms / launches: host pointers, may be NULL. */
int ledds_profile_read(int kernel_id, double* total_ms, int* launches);
/* Number of CUDA kernels launched by this library since it was loaded. */
unsigned long long ledds_launch_count(void);

/* Library version string (host). */
const char* ledds_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LEDDS_H */
