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

// Real type of the DEM path: double on the path of the configs; float = the ledds_dem_*_f32 calls (state, records,
// history and all arithmetic of the step in single precision).
template <typename T> struct Real;
template <> struct Real<double> {
    typedef double4 v4; typedef double2 v2;
    static __host__ __device__ __forceinline__ v4 make4(double a, double b, double c, double d) { return make_double4(a, b, c, d); }
    static __host__ __device__ constexpr double touch_eps() { return 1e-14; }   // |d^2 / (R_i + R_j)^2 - 1| below which Eq. (2) takes the square root
};
template <> struct Real<float> {
    typedef float4 v4; typedef float2 v2;
    static __host__ __device__ __forceinline__ v4 make4(float a, float b, float c, float d) { return make_float4(a, b, c, d); }
    static __host__ __device__ constexpr float touch_eps() { return 1e-6f; }
};

// Kernel-side DEM parameters (passed by value), in the real type of the kernels.
template <typename T>
struct DemDevT {
    int n;
    T lo[3], hi[3], L[3];
    float Lf[3], fmargin;          // single-precision first look of the detect kernel: (float)L, 2^-19 max L
    int bc[3];
    T vw[18];
    int nc[3];
    T inv_h[3];
    unsigned ncell, plane;         // cells in the grid, in one z-plane
    unsigned long long magic_row, magic_plane;   // ceil(2^40 / nc[0]), ceil(2^40 / plane): key decode without divisions
    int magic_ok;
    T hmin;                        // smallest cell width of the grid: 2 R must not exceed it (LEDDS_ST_RADIUS_RANGE)
    T dt, g[3], density;
    T kn, kt, zeta, mu;
    T kn_w, kt_w, zeta_w, mu_w;
    T Ystar, Gstar, Ystar_w, Gstar_w;   // Hertz-Mindlin (A.6), (A.7): sphere-sphere / sphere-wall
    int maxc;
};
typedef DemDevT<double> DemDev;

// Layout of the caller-owned DEM scratch buffer (byte offsets, all 256-B aligned).
// "home" order: the order the library keeps the particle state in between the steps of one call.  It is the
// sorted order (by cell key, then id) of the last sort before the call began, so a particle's home index stays
// close to its sorted position and every access "by particle" is nearly sequential.  The caller's arrays are
// read once when a call begins (import) and written once when it ends (export).
struct DemScratch {
    size_t hist_digit;             // global digit histograms (uint32 [4][256])           } zeroed
    size_t tile_counter;           // dynamic tile tickets of the sort passes and the scan } before
    size_t tile_state;             // look-back descriptors of the sort (uint32 [4][tiles][256]) } every
    size_t scan_state;             // look-back descriptors of the scan (uint32 [scan tiles])    } step
    size_t cell_scan_state;        // look-back descriptors of the scan over the cells (counting sort; zeroed too)
    size_t cell_range;             // uint2 [ncell]: [start, end) of the cell in the sorted order, 0,0 when empty (zeroed too)
    size_t key[2], idx[2];         // ping-pong sort buffers: cell key, home index (uint32 [n])
    size_t hid;                    // uint32 [n]: caller's particle id of home slot h
    size_t sid;                    // uint32 [n]: caller's particle id at sorted position s (last sort)
    size_t sid_tmp;                // uint32 [n]: the same before the particles of a cell are put into id order
    size_t skey_f;                 // uint32 [n]: the sorted keys (from the radix passes, or the home keys when those were skipped)
    size_t hx;                     // double4 [n]: (x, y, z, R), home order
    size_t hv, hw, ha, hal;        // double [n][3]: v, w, a, alpha, home order
    size_t pvw;                    // double [n][6]: predictor (v^p, w^p), home order
    size_t xr_s;                   // double4 [n]: (x, y, z, R), sorted order
    size_t xf_s;                   // float4 [n]: (x - lo, R) in single precision, sorted order (first look only)
    size_t nfwd, nback;            // uint32 [n]: partners a particle found itself / partners that found it (sorted position)
    size_t cand;                   // uint32 [maxc][n]: column s = its partners, found-by-itself from the top, found-by-others from the bottom
    size_t off;                    // uint32 [n + 1]: first contact end of sorted position s (CSR offsets)
    size_t end_s, end_t;           // uint32 [n maxc]: owner (sorted position) and partner (sorted position or wall code) per end
    size_t end_hs, end_ht;         // uint32 [n maxc]: their home indices
    size_t end_prev;               // uint32 [n maxc]: the end of last step this one continues (or none)
    size_t pair_count, pair_off, pos_of_id;   // query scratch (uint32 [n+1])
    size_t total;
};

// Caller-owned DEM history buffer: what one force evaluation leaves for the next.
struct DemHistory {
    size_t fm[2];                  // double [n][6]: contact force and torque per particle, home order (two copies: re-homing permutes)
    size_t row[2];                 // uint2 [n]: (first end, number of ends) of the particle's contacts in hq / hdt, home order
    size_t hq[2];                  // uint32 [n maxc]: partner id per contact end, two generations
    size_t hdt[2];                 // double [n maxc][3]: delta_t per contact end as seen from its owner, two generations
    size_t total;
};

struct ledds_dem {
    ledds_dem_params p;
    DemDev d;                      // parameters in double (host logic reads these whatever the precision)
    DemDevT<float> df;             // the same in float, for the kernels of an fp32 handle
    bool f32;                      // the handle's real type: ledds_dem_*_f32 calls only / fp64 calls only
    DemScratch s;
    DemHistory hs;
    int cur;                       // which generation of hq / hdt holds the latest contacts
    int rec;                       // which copy of fm / row is current
    int sorted_buf;                // which key ping-pong buffer holds the sorted keys
    int sh_buf;                    // which idx ping-pong buffer holds the home index of every sorted position
    bool have_sort;                // sid / idx[sorted_buf] describe a sort of the current particle set
    int key_bits, passes, tiles, scan_tiles, cell_tiles;
    bool counting;                 // order by cell from counting (ncell <= 4 n) instead of radix passes
    long long steps;
    bool small_cells_clear;        // single-launch step: cell_range is all-empty (every step leaves it so)
    // fork/join of the contact pipeline beside the lattice kernels of a coupled step (host resources, lazily made)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
};

// entry points implemented in dem.cu and used by coupled.cu
template <typename T> struct DemKickT { const T* f_ext; const T* m_ext; };   // external force / torque of a kick, [n][3] by caller id, or NULL
typedef DemKickT<double> DemKick;
// caller's arrays -> home order (begins a call); a / alpha may be NULL (zeros)
int ledds_dem_import(ledds_dem* h, const double* x, const double* v, const double* w, const double* a, const double* alpha,
                     const double* radius, void* history, void* scratch, cudaStream_t st);
// home order -> caller's arrays (ends a call); any pointer may be NULL (not written)
int ledds_dem_export(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha, const void* scratch, cudaStream_t st);
// one force evaluation on the home state: [kick of the previous step] -> drift (optional) -> keys -> sort -> contacts
int ledds_dem_advance_contacts(ledds_dem* h, void* history, void* scratch, int32_t* status, double dt_hist,
                               bool drift, cudaStream_t st, bool fork = false, const DemKick* kick = nullptr);
int ledds_dem_kick(ledds_dem* h, const double* f_ext, const double* m_ext, const void* history, void* scratch, cudaStream_t st);
