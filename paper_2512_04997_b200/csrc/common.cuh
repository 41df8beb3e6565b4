// Shared declarations of the CUDA path (sm_100a).  Not used by, and shares nothing with, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/ledds.h"

#define LEDDS_Q 19

// kernel groups for ledds_profile_read (include/ledds.h LEDDS_K_*)
#define LEDDS_K_COUNT 8
void ledds_count_launch(int n);
void ledds_prof_start(int kernel_id, cudaStream_t st);
void ledds_prof_stop(int kernel_id, cudaStream_t st);

// after every kernel launch: count it and surface launch errors
#define LEDDS_CHECK_LAUNCH()                                  \
    do {                                                      \
        ledds_count_launch(1);                                \
        if (cudaPeekAtLastError() != cudaSuccess) return LEDDS_ECUDA; \
    } while (0)

int ledds_sm_count();   // multiprocessors of the current device (cached; prof.cu)

static inline bool ledds_aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ---- D3Q19 tables (numbering of include/ledds.h); constexpr so unrolled loops fold them ----
__host__ __device__ constexpr int lb_cx(int q)
{
    constexpr int t[LEDDS_Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
    return t[q];
}
__host__ __device__ constexpr int lb_cy(int q)
{
    constexpr int t[LEDDS_Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
    return t[q];
}
__host__ __device__ constexpr int lb_cz(int q)
{
    constexpr int t[LEDDS_Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
    return t[q];
}
__host__ __device__ constexpr int lb_opp(int q) { return q == 0 ? 0 : ((q & 1) ? q + 1 : q - 1); }
__host__ __device__ constexpr double lb_w(int q) { return q == 0 ? 1.0 / 3.0 : (q <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }

// Kernel-side view of the lattice parameters (passed by value).
struct LbmDev {
    int nx, ny, nz;
    long long N;
    double omega;          // dt / tau (tau^+ for TRT)
    double omega_minus;    // dt / tau^-, Eq. (31)
    int trt;               // collision model: 0 BGK, 1 TRT
    double tau;
    int bc[3];
    double uw[18];         // [axis][side][comp]
    int any_wall_velocity;
};

struct ledds_lbm {
    ledds_lbm_params p;
    LbmDev d;
    int parity;            // which half of the two-lattice buffer is current (0 or 1)
    long long steps;
    bool f32;              // populations are float (ledds_lbm_*_f32 calls); the coupled step takes fp64 handles only
};

// Kernel-side DEM parameters.
struct DemDev {
    int n;
    double lo[3], hi[3], L[3];
    float Lf[3], fmargin;          // single-precision first look of the detect kernel: (float)L, 2^-19 max L
    int bc[3];
    double vw[18];
    int nc[3];
    double inv_h[3];
    unsigned ncell;
    double hmin;                   // smallest cell width of the grid: 2 R must not exceed it (LEDDS_ST_RADIUS_RANGE)
    double dt, g[3], density;
    double kn, kt, zeta, mu;
    double kn_w, kt_w, zeta_w, mu_w;
    double Ystar, Gstar, Ystar_w, Gstar_w;   // Hertz-Mindlin (A.6), (A.7): sphere-sphere / sphere-wall
    int maxc;
};

// Layout of the caller-owned DEM scratch buffer (byte offsets, all 256-B aligned).
struct DemScratch {
    size_t key[2], idx[2];         // ping-pong sort buffers (uint32 [n])
    size_t hist_digit;             // global digit histograms (uint32 [4][256])
    size_t tile_state;             // look-back descriptors (uint32 [tiles][256])
    size_t tile_counter;           // dynamic tile ticket (uint32 [4])
    size_t cell_range;             // uint2 [ncell]: [start, end) of the cell in the sorted order, 0,0 when empty
    size_t xr, xr_s;               // (x, y, z, R) per particle, 32 B: particle order / sorted order
    size_t xf_s;                   // (x - lo, R) in single precision, sorted order, 16 B (first look only)
    size_t ncand, cand;            // contacts found per sorted position: uint32 [n], uint32 [maxc][n]
    size_t vp, wp;                 // predictor velocities in particle order: double [n][3]
    size_t vw_s;                   // (v^p, w^p) of the particles in contact, sorted order: double [n][6]
    size_t pair_count, pair_off;   // query scratch (uint32 [n+1])
    size_t total;
};

struct DemHistory {
    size_t ft[2];                  // per particle, 64 B: contact force[3], torque[3], number of contacts, history row
    size_t id[2];                  // uint32 [n][maxc], rows in the sorted order of the step that wrote them
    size_t dt[2];                  // double [n][maxc][3], same rows
    size_t total;
};

struct ledds_dem {
    ledds_dem_params p;
    DemDev d;
    DemScratch s;
    DemHistory hs;
    int cur;                       // which history buffer holds the latest contacts
    int sorted_buf;                // which key/idx ping-pong buffer holds the sorted result
    int key_bits, passes, tiles;
    long long steps;
    // fork/join of the contact pipeline beside the lattice kernels of a coupled step (host resources, lazily made)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
};

// entry points implemented in dem.cu and used by coupled.cu
struct DemKick { const double* f_ext; const double* m_ext; };   // external force / torque of a kick, [n][3] or NULL
int ledds_dem_advance_contacts(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha,
                               const double* radius, void* history, void* scratch, int32_t* status, double dt_hist,
                               bool drift, cudaStream_t st, bool fork = false, const DemKick* kick = nullptr);
int ledds_dem_kick(ledds_dem* h, double* v, double* w, double* a, double* alpha, const double* radius,
                   const double* f_ext, const double* m_ext, const void* history, int32_t* status, cudaStream_t st);
