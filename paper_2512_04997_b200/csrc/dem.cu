// DEM contact pipeline for spheres on sm_100a (Eq. 1-15, 158-192 Eq. 18-21, 431-511).
//
// The particle state lives in the library's own "home" order between the steps of one call: the sorted order (cell
// key, then id) of the last sort before the call began.  The caller's arrays are gathered once when a call begins
// (dem_import_kernel) and scattered back once when it ends (dem_export_kernel); in between every per-particle access
// is (nearly) sequential whatever order the caller numbers its particles in.
//
//   dem_drift_key_kernel   [kick of the previous step] + Eq. (18a) + predictor, cell key      (map N_part, home order)
//   dem_hist_kernel        digit histograms of all radix passes in one sweep                  (smem histograms)
//   dem_onesweep_kernel    one stable 8-bit radix pass: per-warp match ranking, chained scan with
//                          decoupled look-back across tiles, scatter                            (x passes)
//   dem_ranges_kernel      cell start/end from the key changes
//   dem_gather_kernel      ties of the sort put into id order; sorted copy of (x, R) + its single-precision copy, ids
//   dem_detect_kernel      every pair of the 27-cell neighbourhood is tested ONCE, from the particle that comes first in
//                          the sorted order (Eq. 2/6 in double after a first look in single precision); a contact is
//                          entered into the lists of both partners (integer atomics on the list lengths)
//   dem_scan_kernel        exclusive scan of the list lengths: the contact ends of all particles as one CSR array
//   dem_fill_kernel        each particle orders its ends by partner id (the order of the paper's sorted pair list)
//   dem_force_kernel       ONE THREAD PER CONTACT END: Eq. (7), (10)-(13), (5), (15), history carried per end; the
//                          per-particle sums of Eq. (1) are taken by the particle's own thread from the block's shared
//                          memory, in the order of the list: no floating-point atomics, bit-reproducible
//   dem_kick_kernel        Eq. (18b-c), (19c-d) for spheres
//
// Compiled with -fmad=false: the discrete decisions (cell index, delta_n > 0) must not depend on
// FMA contraction.  No Thrust/CUB; no global fp atomics.
#include <math.h>

#include <algorithm>
#include <new>

#include "common.cuh"

#define DEM_PI 3.14159265358979323846
#define SORT_THREADS 256
#define SORT_WARPS (SORT_THREADS / 32)
#define SORT_ITEMS 12
#define SORT_MIN_BLOCKS 4
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
#define SORT_RADIX 256

#define ST_FLAG_AGG 0x40000000u
#define ST_FLAG_PRE 0x80000000u
#define ST_VALUE_MASK 0x3fffffffu
#define LOOKBACK 8

#define SCAN_THREADS 256
#define SCAN_ITEMS 16            // per thread: 4 096 values per tile, staged in shared memory so that loads and stores are coalesced
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

#define DEM_WALL 0xfffffff0u    // partner code of wall wl (0..5) in the contact lists: DEM_WALL + wl

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// Programmatic dependent launch: the kernels of a step form one dependent chain of short launches (for a few thousand
// particles each runs a few microseconds).  Every kernel of the chain lets its successor be launched as soon as all of
// its own blocks have started, and waits for its predecessor's results before it touches them: the launch latency of
// kernel k + 1 is hidden behind kernel k.  Used for systems of up to DEM_PDL_MAX_N particles: with millions of particles
// the early-launched blocks only take resident slots from the kernel they wait for (4 M spheres: + 3 %).
#define DEM_PDL_MAX_N 262144
#define DEM_PDL_ENTER(n)                                                \
    do {                                                                \
        if ((n) <= DEM_PDL_MAX_N) {                                     \
            asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); \
            asm volatile("griddepcontrol.wait;" ::: "memory");           \
        }                                                               \
    } while (0)

static thread_local bool g_pdl = false;   // set by dem_advance_t for the launches of one step

template <typename... KArgs, typename... Args>
static void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = g_pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <typename T>
__device__ __forceinline__ T dem_mass(const DemDevT<T>& P, T R) { return P.density * (T(4.0) / T(3.0)) * T(DEM_PI) * R * R * R; }

// num / den for a numerator that is often exactly zero (the force on a particle without a contact): 0 / x sends the whole
// warp through the slow path of the division, so a zero numerator divides a stand-in value and the result is replaced by
// zero; every other numerator gives exactly num / den.  Used where latency counts (the single-launch step of small
// systems: + 1 %); in the bandwidth-bound drift kernel of large systems the extra selects cost more than they save.
template <typename T>
__device__ __forceinline__ T dem_div0(T num, T den)
{
    const bool z = num == T(0.0);
    const T q = (z ? T(1.0) : num) / den;
    return z ? T(0.0) : q;
}

// ------------------------------------------------------------------------------ import / export
// Block = DRIFT_BLOCK particles; the [n][3] arrays are walked as flat arrays (element e = 3 h + k).
#define DRIFT_BLOCK 128

// hid_src: the caller id of every home slot of the NEW home order (NULL: identity).  perm: the OLD home index of the
// particle in new slot h (NULL: identity); the per-particle records of the last force evaluation move with it.
template <typename T>
__global__ void __launch_bounds__(DRIFT_BLOCK) dem_import_kernel(
    int n, const uint32_t* __restrict__ hid_src, const uint32_t* __restrict__ perm, const T* __restrict__ x,
    const T* __restrict__ v, const T* __restrict__ w, const T* __restrict__ a, const T* __restrict__ alpha,
    const T* __restrict__ radius, uint32_t* __restrict__ hid, typename Real<T>::v4* __restrict__ hx, T* __restrict__ hv,
    T* __restrict__ hw, T* __restrict__ ha, T* __restrict__ hal, const T* __restrict__ fm_old,
    const uint2* __restrict__ row_old, T* __restrict__ fm_new, uint2* __restrict__ row_new)
{
    const long long e0 = (long long)blockIdx.x * (3 * DRIFT_BLOCK), ne = 3ll * n;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const long long e = e0 + threadIdx.x + j * DRIFT_BLOCK;
        if (e >= ne) break;
        const int h = (int)(e / 3), k = (int)(e - 3ll * h);
        const size_t src = 3 * (size_t)(hid_src ? hid_src[h] : (uint32_t)h) + k;
        hv[e] = v[src]; hw[e] = w[src];
        ha[e] = a ? a[src] : T(0.0); hal[e] = alpha ? alpha[src] : T(0.0);
    }
    const int h = blockIdx.x * DRIFT_BLOCK + threadIdx.x;
    if (h >= n) return;
    const uint32_t i = hid_src ? hid_src[h] : (uint32_t)h;
    hx[h] = Real<T>::make4(x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2], radius[i]);
    hid[h] = i;
    const size_t o = perm ? perm[h] : (uint32_t)h;
    row_new[h] = row_old[o];
#pragma unroll
    for (int c = 0; c < 6; ++c) fm_new[6 * (size_t)h + c] = fm_old[6 * o + c];
}

template <typename T>
__global__ void __launch_bounds__(DRIFT_BLOCK) dem_export_kernel(
    int n, const uint32_t* __restrict__ hid, const typename Real<T>::v4* __restrict__ hx, const T* __restrict__ hv,
    const T* __restrict__ hw, const T* __restrict__ ha, const T* __restrict__ hal, T* __restrict__ x,
    T* __restrict__ v, T* __restrict__ w, T* __restrict__ a, T* __restrict__ alpha)
{
    const long long e0 = (long long)blockIdx.x * (3 * DRIFT_BLOCK), ne = 3ll * n;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const long long e = e0 + threadIdx.x + j * DRIFT_BLOCK;
        if (e >= ne) break;
        const int h = (int)(e / 3), k = (int)(e - 3ll * h);
        const size_t dst = 3 * (size_t)hid[h] + k;
        if (v) v[dst] = hv[e];
        if (w) w[dst] = hw[e];
        if (a) a[dst] = ha[e];
        if (alpha) alpha[dst] = hal[e];
    }
    const int h = blockIdx.x * DRIFT_BLOCK + threadIdx.x;
    if (h >= n || !x) return;
    const typename Real<T>::v4 r = hx[h];
    const size_t i = hid[h];
    x[3 * i] = r.x; x[3 * i + 1] = r.y; x[3 * i + 2] = r.z;
}

// ------------------------------------------------------------------------------ drift + key
template <typename T>
__device__ __forceinline__ int dem_cell_coord(const DemDevT<T>& P, T x, int a)
{
    int c = (int)floor((x - P.lo[a]) * P.inv_h[a]);
    c = c < 0 ? 0 : c;
    return c > P.nc[a] - 1 ? P.nc[a] - 1 : c;
}

// KICK = true: the kick of the previous step (Eq. 18b-c, 19c-d with the contact sums fm and the external force /
// torque, which the caller indexes by particle id) is applied first, in the same pass: between two steps of one call
// the state is read and written once instead of twice.  The new velocities and accelerations pass through shared
// memory to the thread that owns the particle's packed (x, R) record.
template <typename T, bool KICK>
__global__ void __launch_bounds__(DRIFT_BLOCK) dem_drift_key_kernel(
    const DemDevT<T> P, typename Real<T>::v4* __restrict__ hx, T* __restrict__ hv, T* __restrict__ hw, T* __restrict__ ha,
    T* __restrict__ hal, const uint32_t* __restrict__ hid, const T* __restrict__ fm,
    const T* __restrict__ f_ext, const T* __restrict__ m_ext, T* __restrict__ pvw,
    uint32_t* __restrict__ key, uint32_t* __restrict__ idx, int drift, int32_t* __restrict__ status,
    uint2* __restrict__ cells /* counting sort: .y of a cell counts its particles (NULL: radix sort, idx = home index) */)
{
    __shared__ T sv[3 * DRIFT_BLOCK], sa[3 * DRIFT_BLOCK];
    const long long e0 = (long long)blockIdx.x * (3 * DRIFT_BLOCK), ne = 3ll * P.n;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int le = threadIdx.x + j * DRIFT_BLOCK;
        const long long e = e0 + le;
        if (e >= ne) break;
        const int h = (int)(e / 3), k = le % 3;                               // e0 is a multiple of 3
        T vv = hv[e], wv = hw[e], av = ha[e], alv = hal[e];
        if (KICK) {                                                           // same expressions as dem_kick_kernel
            const T R = reinterpret_cast<const T*>(hx)[4 * (size_t)h + 3];
            const T m = dem_mass(P, R), I = T(0.4) * m * R * R;             // Eq. (21a)
            const size_t ie = (f_ext || m_ext) ? 3 * (size_t)hid[h] + k : 0;
            const T Fq = fm[6 * (size_t)h + k] + (f_ext ? f_ext[ie] : T(0.0)), Mq = fm[6 * (size_t)h + 3 + k] + (m_ext ? m_ext[ie] : T(0.0));
            const T an = Fq / m + P.g[k], aln = Mq / I;                  // Eq. (18b), (19c)
            vv = vv + (T(0.5) * P.dt) * (av + an);                               // Eq. (18c)
            wv = wv + (T(0.5) * P.dt) * (alv + aln);                             // Eq. (19d)
            av = an; alv = aln;
            hv[e] = vv; hw[e] = wv; ha[e] = av; hal[e] = alv;
        }
        if (drift) {
            pvw[6 * (size_t)h + k] = vv + (T(0.5) * P.dt) * av;                  // predictor (G11)
            pvw[6 * (size_t)h + 3 + k] = wv + (T(0.5) * P.dt) * alv;
        } else {
            pvw[6 * (size_t)h + k] = vv;
            pvw[6 * (size_t)h + 3 + k] = wv;
        }
        sv[le] = vv; sa[le] = av;
    }
    __syncthreads();
    const int h = blockIdx.x * DRIFT_BLOCK + threadIdx.x;
    if (h >= P.n) return;
    const typename Real<T>::v4 r = hx[h];
    T xn[3] = {r.x, r.y, r.z};
    if (drift) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            T xv = xn[k] + P.dt * sv[3 * threadIdx.x + k] + (T(0.5) * P.dt * P.dt) * sa[3 * threadIdx.x + k];   // Eq. (18a)
            if (!P.bc[k]) {
                if (xv >= P.hi[k]) xv -= P.L[k];
                else if (xv < P.lo[k]) xv += P.L[k];
            }
            xn[k] = xv;
        }
        hx[h] = Real<T>::make4(xn[0], xn[1], xn[2], r.w);
    }
    const int cx = dem_cell_coord(P, xn[0], 0), cy = dem_cell_coord(P, xn[1], 1), cz = dem_cell_coord(P, xn[2], 2);
    const uint32_t ck = (uint32_t)(cx + P.nc[0] * (cy + P.nc[1] * cz));
    key[h] = ck;
    idx[h] = cells ? atomicAdd(&cells[ck].y, 1u) : (uint32_t)h;                  // its number among the particles of its cell
    // input contract (include/ledds.h): 2 R <= cell width, centres inside a walled box
    int st = T(2.0) * r.w > P.hmin ? LEDDS_ST_RADIUS_RANGE : 0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (P.bc[a] && !(xn[a] >= P.lo[a] && xn[a] <= P.hi[a])) st |= LEDDS_ST_OUT_OF_BOX;
    if (st) atomicOr(status, st);
}

// key -> (cx, cy, cz).  The two divisions by run-time constants are multiplications by host-computed reciprocals:
// floor(k m / 2^40) with m = ceil(2^40 / d) equals floor(k / d) whenever k d <= 2^40 (the host checks it for the
// largest key and both divisors; else the plain divisions are used).
template <typename T>
__device__ __forceinline__ void dem_cell_of_key(const DemDevT<T>& P, uint32_t key, int& c0, int& c1, int& c2)
{
    uint32_t r, z;
    if (P.magic_ok) {
        z = (uint32_t)(((unsigned long long)key * P.magic_plane) >> 40);
        const uint32_t rem = key - z * P.plane;
        r = (uint32_t)(((unsigned long long)rem * P.magic_row) >> 40);
        c0 = (int)(rem - r * (uint32_t)P.nc[0]);
    } else {
        z = key / P.plane;
        const uint32_t rem = key - z * P.plane;
        r = rem / (uint32_t)P.nc[0];
        c0 = (int)(rem - r * (uint32_t)P.nc[0]);
    }
    c1 = (int)r; c2 = (int)z;
}

// ------------------------------------------------------------------------------ radix sort
// All digit histograms in one pass over the keys (smem atomics, then one global add per bin).  The keys arrive in
// home order, i.e. nearly sorted: the upper digits of a warp's 32 keys are usually all the same, and one lane then
// adds 32 instead of 32 lanes queueing on one shared-memory word.  The same sweep checks whether the keys are still in
// non-descending order: then this step's sort is the identity (ties inside a cell are put into id order by
// dem_gather_kernel in any case) and the radix passes return at once -- the rule in a settled bed, where a particle
// changes its cell once in thousands of steps (the paper's own cell lists are updated incrementally on the same
// grounds).  ledds_dem_params.sort_every_step = 1 switches that off (measurement).
__global__ void __launch_bounds__(SORT_THREADS) dem_hist_kernel(const uint32_t* __restrict__ key, int n, int passes,
                                                               uint32_t* __restrict__ ghist, uint32_t* __restrict__ unsorted)
{
    DEM_PDL_ENTER(n);
    __shared__ uint32_t h[4][SORT_RADIX];
    for (int t = threadIdx.x; t < 4 * SORT_RADIX; t += blockDim.x) (&h[0][0])[t] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int per = ((n + 127) / 128 + gridDim.x - 1) / gridDim.x * 128;          // a contiguous piece per block, 4 keys per lane and round
    const int beg = blockIdx.x * per, end = min(n, beg + per);
    for (int base = beg + (threadIdx.x & ~31) * 4; base < end; base += blockDim.x * 4) {
        uint32_t k4[4];
        bool ok4[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {                                             // four independent loads in flight
            const int i = base + j * 32 + lane;
            ok4[j] = i < end;
            k4[j] = ok4[j] ? key[i] : 0u;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool ok = ok4[j];
            const uint32_t k = k4[j];
            const unsigned live = __ballot_sync(0xffffffffu, ok);
            if (!live) continue;
            {   // are the keys still in order (home order = last sorted order)?  Then the sort of this step is the identity.
                const int i = base + j * 32 + lane;
                uint32_t pk = __shfl_up_sync(0xffffffffu, k, 1);
                if (lane == 0) pk = i > 0 ? key[i - 1] : 0u;
                if (ok && k < pk) *unsorted = 1u;
            }
            for (int p = 0; p < passes; ++p) {
                const uint32_t d = (k >> (8 * p)) & 255u;
                const uint32_t d0 = __shfl_sync(0xffffffffu, d, __ffs(live) - 1);
                if (__all_sync(0xffffffffu, !ok || d == d0)) {
                    if (lane == 0) atomicAdd(&h[p][d0], (uint32_t)__popc(live));
                } else if (ok) {
                    atomicAdd(&h[p][d], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < passes * SORT_RADIX; t += blockDim.x) {
        const uint32_t c = (&h[0][0])[t];
        if (c) atomicAdd(&ghist[t], c);
    }
}

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v) { *reinterpret_cast<volatile uint32_t*>(p) = v; }

// One stable LSD pass (8-bit digit at `shift`).  Tiles take tickets from an atomic counter so that
// every tile a block waits on is already resident or done.  Order inside a tile = (warp, item, lane)
// = ascending input index, which keeps the sort stable.
__global__ void __launch_bounds__(SORT_THREADS, SORT_MIN_BLOCKS) dem_onesweep_kernel(
    const uint32_t* __restrict__ key_in, const uint32_t* __restrict__ val_in, uint32_t* __restrict__ key_out,
    uint32_t* __restrict__ val_out, int n, int shift, const uint32_t* __restrict__ ghist /*[256] of this pass*/,
    uint32_t* __restrict__ tile_state /*[tiles][256] of this pass*/, uint32_t* __restrict__ ticket,
    const uint32_t* __restrict__ unsorted, int always)
{
    DEM_PDL_ENTER(n);
    if (!always && *unsorted == 0u) return;                     // the keys are in order already (block-uniform)
    __shared__ uint32_t warp_hist[SORT_WARPS][SORT_RADIX];
    __shared__ uint32_t bin_base[SORT_RADIX];
    __shared__ uint32_t tile_start[SORT_RADIX];
    __shared__ uint32_t wsum2[SORT_WARPS];
    __shared__ uint32_t stage_key[SORT_TILE], stage_val[SORT_TILE];
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int t = tid; t < SORT_WARPS * SORT_RADIX; t += SORT_THREADS) (&warp_hist[0][0])[t] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;

    // exclusive prefix of the global digit histogram (thread d owns digit d)
    uint32_t digit_excl;
    {
        const uint32_t c = ghist[tid];
        uint32_t incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        __shared__ uint32_t wsum[SORT_WARPS];
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t base = 0;
        for (int w2 = 0; w2 < warp; ++w2) base += wsum[w2];
        digit_excl = base + incl - c;
    }

    // load (warp-striped) and rank inside the warp
    uint32_t k[SORT_ITEMS], v[SORT_ITEMS], r[SORT_ITEMS];
    const long long base = (long long)tile * SORT_TILE + (long long)warp * (SORT_ITEMS * 32);
#pragma unroll
    for (int it = 0; it < SORT_ITEMS; ++it) {                   // all loads first: 2 x SORT_ITEMS independent requests
        const long long i = base + it * 32 + lane;
        const bool ok = i < n;
        k[it] = ok ? key_in[i] : 0xffffffffu;
        v[it] = ok ? val_in[i] : 0u;
    }
#pragma unroll
    for (int it = 0; it < SORT_ITEMS; ++it) {
        const bool ok = base + it * 32 + lane < n;
        const uint32_t d = ok ? ((k[it] >> shift) & 255u) : 256u;
        uint32_t peers = 0xffffffffu;                               // lanes with the same digit: 9 ballots, one per bit
#pragma unroll
        for (int b = 0; b < 9; ++b) {
            const bool bit = (d >> b) & 1u;
            const uint32_t bal = __ballot_sync(0xffffffffu, bit);
            peers &= bit ? bal : ~bal;
        }
        const uint32_t below = __popc(peers & ((1u << lane) - 1u));
        uint32_t old = 0;
        if (ok) old = warp_hist[warp][d];
        __syncwarp();
        if (ok && below == 0) warp_hist[warp][d] = old + __popc(peers);
        __syncwarp();
        r[it] = old + below;
    }
    __syncthreads();

    // per digit: exclusive scan over the warps of this tile, then the chained scan over tiles
    {
        const int d = tid;
        uint32_t run = 0;
#pragma unroll
        for (int w2 = 0; w2 < SORT_WARPS; ++w2) {
            const uint32_t c = warp_hist[w2][d];
            warp_hist[w2][d] = run;
            run += c;
        }
        uint32_t* my = tile_state + (size_t)tile * SORT_RADIX + d;
        uint32_t excl = 0;
        if (tile == 0) {
            st_volatile(my, ST_FLAG_PRE | run);
        } else {
            st_volatile(my, ST_FLAG_AGG | run);
            // look back over the predecessors' descriptors, LOOKBACK of them per round trip
            long long t = (long long)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t sv[LOOKBACK];
#pragma unroll
                for (int b = 0; b < LOOKBACK; ++b)
                    sv[b] = t - b >= 0 ? ld_volatile(tile_state + (size_t)(t - b) * SORT_RADIX + d) : ST_FLAG_PRE;
#pragma unroll
                for (int b = 0; b < LOOKBACK; ++b) {
                    if (done) break;
                    uint32_t sb = sv[b];
                    while ((sb & (ST_FLAG_AGG | ST_FLAG_PRE)) == 0) sb = ld_volatile(tile_state + (size_t)(t - b) * SORT_RADIX + d);
                    excl += sb & ST_VALUE_MASK;
                    if (sb & ST_FLAG_PRE) done = true;
                }
                t -= LOOKBACK;
            }
            st_volatile(my, ST_FLAG_PRE | (excl + run));
        }
        // where digit d starts inside this tile once the tile is ordered by digit (block-wide exclusive scan of run)
        uint32_t incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) wsum2[warp] = incl;
        __syncthreads();
        uint32_t before = 0;
        for (int w2 = 0; w2 < warp; ++w2) before += wsum2[w2];
        tile_start[d] = before + incl - run;
        bin_base[d] = digit_excl + excl - (before + incl - run);    // global position = bin_base[d] + position in the tile
    }
    __syncthreads();

    // order the tile by digit in shared memory, so that the global writes of a digit are contiguous
#pragma unroll
    for (int it = 0; it < SORT_ITEMS; ++it) {
        if (base + it * 32 + lane < n) {
            const uint32_t d = (k[it] >> shift) & 255u;
            const uint32_t lp = tile_start[d] + warp_hist[warp][d] + r[it];
            stage_key[lp] = k[it];
            stage_val[lp] = v[it];
        }
    }
    __syncthreads();
    const long long tile_first = (long long)tile * SORT_TILE;
    const int count = (int)min((long long)SORT_TILE, (long long)n - tile_first);
    for (int i = tid; i < count; i += SORT_THREADS) {
        const uint32_t kk = stage_key[i];
        const uint32_t dst = bin_base[(kk >> shift) & 255u] + (uint32_t)i;
        key_out[dst] = kk;
        val_out[dst] = stage_val[i];
    }
}

// ------------------------------------------------------------------------------ counting sort
// When the grid has about as many cells as there are particles (a packed bed, a pour: ncell <= 4 n) the order by cell
// comes cheaper from counting than from radix passes over the keys: every particle has counted itself into its cell
// in the drift kernel (integer atomic, the returned value is its number inside the cell), one chained scan over the
// CELLS turns the counts into [start, end) -- which is the cell-range table itself, no pass over sorted keys needed
// -- and one scatter puts (key, home index, id) at start + number.  The order inside a cell is the order of arrival
// here; dem_gather_kernel ranks the particles of a cell by id as it does after the radix sort, so the final order
// (cell key, id) is the same, bit for bit.  Same tile / ticket / look-back scheme as dem_scan_kernel below.
// Chained exclusive scan of one tile of SCAN_TILE values, common to dem_cell_scan_kernel and dem_scan_kernel.  The
// values were put into sc[] (padded index scan_pad(x), so that a thread's SCAN_ITEMS consecutive values and a warp's
// 32 consecutive values are both conflict-free); on return sc[scan_pad(x)] = global exclusive prefix of value x and the
// function's value = global prefix at the end of the tile.  Tiles take tickets (every tile a block waits for is resident
// or done); a tile publishes its sum at once and the first warp looks back over 32 predecessors per round trip.
__device__ __forceinline__ int scan_pad(int x) { return x + (x >> 5); }
#define SCAN_SMEM (SCAN_TILE + SCAN_TILE / 32)

__device__ __forceinline__ uint32_t scan_tile_chained(uint32_t* sc, uint32_t tile, uint32_t* __restrict__ state)
{
    __shared__ uint32_t wsum[SCAN_THREADS / 32];
    __shared__ uint32_t s_excl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t c[SCAN_ITEMS], sum = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { c[i] = sc[scan_pad(tid * SCAN_ITEMS + i)]; sum += c[i]; }
    uint32_t incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t before = 0, total = 0;
#pragma unroll
    for (int w2 = 0; w2 < SCAN_THREADS / 32; ++w2) {
        if (w2 < warp) before += wsum[w2];
        total += wsum[w2];
    }
    if (warp == 0) {
        uint32_t excl = 0;
        if (tile == 0) {
            if (lane == 0) st_volatile(state, ST_FLAG_PRE | total);
        } else {
            if (lane == 0) st_volatile(state + tile, ST_FLAG_AGG | total);
            long long t = (long long)tile - 1;
            for (;;) {
                const long long i = t - lane;
                uint32_t sb = i >= 0 ? ld_volatile(state + i) : ST_FLAG_PRE;
                while (__any_sync(0xffffffffu, (sb & (ST_FLAG_AGG | ST_FLAG_PRE)) == 0))
                    if ((sb & (ST_FLAG_AGG | ST_FLAG_PRE)) == 0) sb = ld_volatile(state + i);
                const unsigned pre = __ballot_sync(0xffffffffu, (sb & ST_FLAG_PRE) != 0);
                const int last = pre ? __ffs(pre) - 1 : 31;                         // the nearest predecessor with a full prefix
                uint32_t v = lane <= last ? (sb & ST_VALUE_MASK) : 0u;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                excl += v;
                if (pre) break;
                t -= 32;
            }
            if (lane == 0) st_volatile(state + tile, ST_FLAG_PRE | (excl + total));
        }
        if (lane == 0) s_excl = excl;
    }
    __syncthreads();
    uint32_t run = s_excl + before + incl - sum;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { sc[scan_pad(tid * SCAN_ITEMS + i)] = run; run += c[i]; }
    __syncthreads();
    return s_excl + total;
}

__global__ void __launch_bounds__(SCAN_THREADS) dem_cell_scan_kernel(int n, uint32_t ncell, uint2* __restrict__ cells,
                                                                    uint32_t* __restrict__ state, uint32_t* __restrict__ ticket)
{
    DEM_PDL_ENTER(n);
    __shared__ uint32_t sc[SCAN_SMEM];
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const long long base = (long long)tile * SCAN_TILE;
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {                                          // coalesced: a warp reads 32 consecutive cells
        const int x = j * SCAN_THREADS + tid;
        sc[scan_pad(x)] = base + x < (long long)ncell ? cells[base + x].y : 0u;
    }
    __syncthreads();
    const uint32_t end = scan_tile_chained(sc, tile, state);
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        const int x = j * SCAN_THREADS + tid;
        const uint32_t start = sc[scan_pad(x)], stop = x + 1 < SCAN_TILE ? sc[scan_pad(x + 1)] : end;
        if (stop > start) cells[base + x] = make_uint2(start, stop);                // an empty cell stays (0, 0)
    }
}

__global__ void dem_scatter_kernel(int n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ slot,
                                   const uint2* __restrict__ cells, const uint32_t* __restrict__ hid,
                                   uint32_t* __restrict__ key_sorted, uint32_t* __restrict__ idx_sorted, uint32_t* __restrict__ sid_tmp)
{
    DEM_PDL_ENTER(n);
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n) return;
    const uint32_t k = key[h];
    const uint32_t p = cells[k].x + slot[h];
    key_sorted[p] = k;
    idx_sorted[p] = (uint32_t)h;
    sid_tmp[p] = hid[h];
}

// ------------------------------------------------------------------------------ cell ranges + gather
// The radix sort is stable with respect to its input order, the home order: inside a cell, particles that were there
// before keep their relative (id) order, but one that has just moved in stands where its old home index puts it.  The
// ordering the pipeline promises is (cell key, then ascending id) -- the stable sort of the ids, PAPER.md:388 -- so the
// particles of a cell are ranked by id once more (cells hold a handful of particles).
//   dem_ranges_kernel: [start, end) of every cell from the key changes (warp shuffle of neighbouring keys), and the id
//                      of every particle in key-sorted order
//   dem_gather_kernel: rank inside the cell by id -> final sorted position; sorted copies of (x, R), ids, home indices
__global__ void dem_ranges_kernel(int n, const uint32_t* __restrict__ key_home, const uint32_t* __restrict__ key_sorted,
                                  const uint32_t* __restrict__ idx_sorted, const uint32_t* __restrict__ unsorted, int always,
                                  const uint32_t* __restrict__ hid, uint32_t* __restrict__ sid_tmp, uint2* __restrict__ cell_range)
{
    DEM_PDL_ENTER(n);
    const bool sorted = always || *unsorted != 0u;              // did the radix passes run?  Else sorted order = home order
    const uint32_t* skey = sorted ? key_sorted : key_home;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool ok = s < n;
    const uint32_t key = ok ? skey[s] : 0xffffffffu;
    // neighbours' keys inside the warp by shuffle, across warps by one extra load
    uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
    uint32_t next = __shfl_down_sync(0xffffffffu, key, 1);
    if (!ok) return;
    if (lane == 0) prev = s > 0 ? skey[s - 1] : 0xffffffffu;
    if (lane == 31 || s == n - 1) next = s < n - 1 ? skey[s + 1] : 0xffffffffu;
    if (s == 0 || prev != key) cell_range[key].x = (uint32_t)s;                    // [x, y) = the particles of the cell
    if (s == n - 1 || next != key) cell_range[key].y = (uint32_t)s + 1u;
    sid_tmp[s] = hid[sorted ? idx_sorted[s] : (uint32_t)s];
}

// idx_sorted[s] = home index of the particle at key-sorted position s (a nearly sequential read of the home records)
template <typename T>
__global__ void dem_gather_kernel(const DemDevT<T> P, const uint32_t* __restrict__ key_home, const uint32_t* __restrict__ key_sorted,
                                  const uint32_t* __restrict__ idx_sorted, const uint32_t* __restrict__ unsorted, int always,
                                  uint32_t* __restrict__ skey_f, const uint32_t* __restrict__ sid_tmp, const uint2* __restrict__ cell_range,
                                  const typename Real<T>::v4* __restrict__ hx, typename Real<T>::v4* __restrict__ xr_s, float4* __restrict__ xf_s,
                                  uint32_t* __restrict__ sid, uint32_t* __restrict__ sh, uint32_t* __restrict__ nback)
{
    DEM_PDL_ENTER(P.n);
    const int s0 = blockIdx.x * blockDim.x + threadIdx.x;
    if (s0 >= P.n) return;
    const bool sorted = always || *unsorted != 0u;
    const uint32_t key = sorted ? key_sorted[s0] : key_home[s0];
    const uint2 cr = cell_range[key];
    const uint32_t id = sid_tmp[s0];
    uint32_t s = cr.x;
    for (uint32_t t = cr.x; t < cr.y; ++t) s += sid_tmp[t] < id;                   // ids are distinct
    const uint32_t h = sorted ? idx_sorted[s0] : (uint32_t)s0;
    skey_f[s] = key;                                                               // the sorted keys, whichever way they came
    const typename Real<T>::v2* src = reinterpret_cast<const typename Real<T>::v2*>(hx + h);
    const typename Real<T>::v2 a = __ldg(src), b = __ldg(src + 1);
    xr_s[s] = Real<T>::make4(a.x, a.y, b.x, b.y);
    sid[s] = id;
    sh[s] = h;
    nback[s] = 0u;
    // single-precision copy (x - lo, R) for the detect kernel's first look at a candidate (dem_near).  A particle
    // further than 2 L from the box corner (or not finite) gets NaN: it passes every first look.
    const T rx = a.x - P.lo[0], ry = a.y - P.lo[1], rz = b.x - P.lo[2];
    const bool sane = fabs(rx) <= T(2.0) * P.L[0] && fabs(ry) <= T(2.0) * P.L[1] && fabs(rz) <= T(2.0) * P.L[2];
    const float qnan = __int_as_float(0x7fc00000);
    xf_s[s] = sane ? make_float4((float)rx, (float)ry, (float)rz, (float)b.y) : make_float4(qnan, qnan, qnan, qnan);
}

// ------------------------------------------------------------------------------ contact law
template <typename T>
__device__ __forceinline__ void cross3(const T* a, const T* b, T* c)
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

// r_i - r_j with the nearest image on periodic axes
template <typename T>
__device__ __forceinline__ void dem_min_image(const DemDevT<T>& P, const T* xi, const T* xj, T* d)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        d[a] = xi[a] - xj[a];
        if (!P.bc[a]) {
            if (d[a] > T(0.5) * P.L[a]) d[a] -= P.L[a];
            else if (d[a] < -T(0.5) * P.L[a]) d[a] += P.L[a];
        }
    }
}

// Force of one contact in its canonical orientation (i < j, or j = wall), Eq. (4)-(15).
// en, dn: unit normal from j to i and overlap.  dt3: in = previous delta_t, out = new delta_t.
// F = force on i; T = e_n x F_t (torque on a body of radius R is -R T, Eq. 15).
template <typename T>
__device__ __forceinline__ void dem_pair_force(const T* en, T dn, const T* vi, const T* wi,
                                               T Ri, const T* vj, const T* wj, T Rj,
                                               T kn, T kt, T gn, T gt, T mu,
                                               T dt_hist, T* dt3, T* F, T* Tq)
{
    T rw[3], rwxe[3], vrel[3], vt[3], Ft[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) rw[a] = Ri * wi[a] + Rj * wj[a];
    cross3(rw, en, rwxe);
#pragma unroll
    for (int a = 0; a < 3; ++a) vrel[a] = (vi[a] - vj[a]) - rwxe[a];                  // Eq. (11)
    const T vn = vrel[0] * en[0] + vrel[1] * en[1] + vrel[2] * en[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) vt[a] = vrel[a] - vn * en[a];                         // Eq. (12)
    const T fn = kn * dn - gn * vn;                                              // Eq. (10)
    const T dte = dt3[0] * en[0] + dt3[1] * en[1] + dt3[2] * en[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) dt3[a] = (dt3[a] - dte * en[a]) + dt_hist * vt[a];    // Eq. (13)
#pragma unroll
    for (int a = 0; a < 3; ++a) Ft[a] = -kt * dt3[a] - gt * vt[a];                    // Eq. (4)
    const T ft = sqrt(Ft[0] * Ft[0] + Ft[1] * Ft[1] + Ft[2] * Ft[2]), fmax = mu * fabs(fn);
    if (ft > fmax) {                                                                  // Eq. (5)
        const T s = fmax / ft;
#pragma unroll
        for (int a = 0; a < 3; ++a) { Ft[a] *= s; dt3[a] = -(Ft[a] + gt * vt[a]) / kt; }
    }
    cross3(en, Ft, Tq);
#pragma unroll
    for (int a = 0; a < 3; ++a) F[a] = fn * en[a] + Ft[a];
}

// Tuning constants (the measured best at 4 M spheres)
#define CONTACT_BLOCK 128       // threads per block of the detect and fill kernels
#define DETECT_NB 3             // candidates in flight per iteration of the detect loop
#define DETECT_MIN_BLOCKS 8     // caps the detect kernel at 64 registers (8 blocks per SM)
#define FORCE_THREADS 128       // one thread per contact end ...
#define FORCE_WARPS (FORCE_THREADS / 32)
#define FORCE_PW 64             // ... of the FORCE_PW particles of a warp: ~7 rounds of 32 ends in a dense bed
#define FORCE_PB (FORCE_WARPS * FORCE_PW)
#define FORCE_MIN_BLOCKS 6

// Stiffness and damping of one contact.  HERTZ = false: the linear spring-dashpot of the configs, gamma =
// 2 zeta sqrt(k m*) (G5).  HERTZ = true: Hertz-Mindlin: (A.1) k_n = 4/3 Y* sqrt(R* d_n),
// k_t = 8 G* sqrt(R* d_n); (A.3)-(A.4) S_n = 2 Y* sqrt(R* d_n), S_t = 8 G* sqrt(R* d_n); (A.2) gamma =
// 2 sqrt(5/6) zeta sqrt(S m*), zeta = -beta of (A.5).  Y*, G* of (A.6)-(A.7) come from the host (one material).
template <typename T, bool HERTZ>
__device__ __forceinline__ void dem_coefficients(T kn0, T kt0, T Ystar, T Gstar, T zeta, T mstar,
                                                 T Rstar, T dn, T& kn, T& kt, T& gn, T& gt)
{
    if (HERTZ) {
        const T sq = sqrt(Rstar * dn);
        kn = (T(4.0) / T(3.0)) * Ystar * sq;
        kt = T(8.0) * Gstar * sq;
        const T Sn = T(2.0) * Ystar * sq, St = T(8.0) * Gstar * sq;
        gn = T(2.0) * sqrt(T(5.0) / T(6.0)) * zeta * sqrt(Sn * mstar);
        gt = T(2.0) * sqrt(T(5.0) / T(6.0)) * zeta * sqrt(St * mstar);
    } else {
        kn = kn0; kt = kt0;
        gn = T(2.0) * zeta * sqrt(kn * mstar); gt = T(2.0) * zeta * sqrt(kt * mstar);
    }
}

// First look at a candidate on the 16-byte single-precision records: false only when the pair is certainly apart.
// Stored coordinates are within 2 L of the origin, so each is off by <= L 2^-23, a difference by <= L 2^-22 (+ the
// rounding of L itself on a wrapped axis) and the distance by < 5e-7 L; fmargin = 2^-19 max L = 1.9e-6 L covers
// that four times over and the factor 1.00001 the roundings of the squares.  NaN records compare as "maybe".
template <typename T, bool PERIODIC>
__device__ __forceinline__ bool dem_near(const DemDevT<T>& P, const float4& a, const float4& b)
{
    float d[3] = {a.x - b.x, a.y - b.y, a.z - b.z};
    if (PERIODIC) {
#pragma unroll
        for (int k = 0; k < 3; ++k)
            if (!P.bc[k]) {
                if (d[k] > 0.5f * P.Lf[k]) d[k] -= P.Lf[k];
                else if (d[k] < -0.5f * P.Lf[k]) d[k] += P.Lf[k];
            }
    }
    const float d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const float lim = (a.w + b.w) + P.fmargin;
    return !(d2 > lim * lim * 1.00001f);
}

// PERIODIC = false: no axis is periodic, the nearest image is the particle itself
template <typename T, bool PERIODIC>
__device__ __forceinline__ bool dem_touch(const DemDevT<T>& P, const typename Real<T>::v4& a, const typename Real<T>::v4& b)
{
    const T xa[3] = {a.x, a.y, a.z}, xb[3] = {b.x, b.y, b.z};
    T d[3] = {xa[0] - xb[0], xa[1] - xb[1], xa[2] - xb[2]};
    if (PERIODIC) dem_min_image(P, xa, xb, d);
    const T d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const T sr = a.w + b.w, s2 = sr * sr;
    if (d2 > s2 * (T(1.0) + Real<T>::touch_eps())) return false;
    if (d2 < s2 * (T(1.0) - Real<T>::touch_eps())) return true;
    return sr - sqrt(d2) > T(0.0);                                                       // Eq. (2), (6), strict (G7)
}

// ------------------------------------------------------------------------------ detect
// One thread per particle in sorted order.  The 9 runs of x-adjacent neighbour cells (contiguous in the sorted order;
// a periodic row adds its one wrapped cell) are loaded up front and clipped to the positions AFTER the particle's own:
// every unordered pair of the neighbourhood is looked at once, from the partner that comes first in the sorted order.
// A contact is entered into both partners' lists: column s of cand[maxc][n] holds, from the top, the partners found by
// the particle itself (sorted positions > s, and DEM_WALL + wall) and, from the bottom, those that found it (arrival order,
// which differs from run to run); dem_fill_kernel puts every list into the order of the partner ids.
// (One thread per (particle, row) -- nine times the threads, a ninth of the work each -- was measured and is slower:
// 0.61 against 0.52 ms in the dense 4 M state, 0.29 against 0.15 ms in the dilute one.)
// The walk of the particle at sorted position s; returns the number of partners it found itself (nfwd[s]), status bits
// are or-ed into st.  nback may be global or shared memory (the single-block step keeps it in shared memory).
template <typename T, bool PERIODIC>
__device__ __forceinline__ uint32_t dem_detect_one(
    const DemDevT<T>& P, const int s, const uint32_t* __restrict__ skey, const typename Real<T>::v4* __restrict__ xr_s,
    const float4* __restrict__ xf_s, const uint2* __restrict__ cell_range, uint32_t* __restrict__ nback,
    uint32_t* __restrict__ cand, int& st)
{
    const uint32_t maxc = (uint32_t)P.maxc;
    const uint32_t key = skey[s];
    const typename Real<T>::v4 mine = xr_s[s];
    const float4 minef = xf_s[s];

    int c0, c1, c2;
    dem_cell_of_key(P, key, c0, c1, c2);

    // A contact (s, t), t > s, goes into two lists.  Mine: slots 0, 1, ... of my column, counted in a register (only this
    // thread writes them).  The partner's: slots maxc-1, maxc-2, ... of its column, the slot taken with an atomic on
    // nback[t]; the store that needs the atomic's result is put off until the next contact (or the end), so the
    // round trip to L2 is covered by the tests in between.
    uint32_t nf = 0, pend_c = 0, pend_t = 0xffffffffu;
    auto flush = [&]() {
        if (pend_t != 0xffffffffu) {
            if (pend_c < maxc) cand[(size_t)(maxc - 1u - pend_c) * P.n + pend_t] = (uint32_t)s;
            else st |= LEDDS_ST_CONTACT_OVERFLOW;
        }
    };
    auto own = [&](uint32_t partner) {
        if (nf < maxc) cand[(size_t)nf * P.n + s] = partner;
        else st |= LEDDS_ST_CONTACT_OVERFLOW;
        ++nf;
    };
    auto enter = [&](uint32_t t) {
        own(t);
        flush();
        pend_c = atomicAdd(nback + t, 1u);
        pend_t = t;
    };
    // the 9 runs [t0, t1) of x-adjacent cells (c0-1 .. c0+1 inside the row): all 27 range loads are independent
    // and issued together; an empty cell holds (0, 0), so "first start, last end" needs no special case
    uint32_t t0[9], t1[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) {
        int qz = c2 + (j / 3 - 1), qy = c1 + (j % 3 - 1);
        bool ok = true;
        if (qz < 0 || qz >= P.nc[2]) { if (P.bc[2]) ok = false; else qz = qz < 0 ? qz + P.nc[2] : qz - P.nc[2]; }
        if (qy < 0 || qy >= P.nc[1]) { if (P.bc[1]) ok = false; else qy = qy < 0 ? qy + P.nc[1] : qy - P.nc[1]; }
        const uint2 none = make_uint2(0u, 0u);
        uint2 r0 = none, r1 = none, r2 = none;
        if (ok) {
            const uint2* row = cell_range + (size_t)P.nc[0] * (size_t)(qy + P.nc[1] * qz) + c0;
            r1 = row[0];
            if (c0 > 0) r0 = row[-1];
            if (c0 < P.nc[0] - 1) r2 = row[1];
        }
        const bool e0 = r0.y > r0.x, e1 = r1.y > r1.x, e2 = r2.y > r2.x;
        t0[j] = max(e0 ? r0.x : (e1 ? r1.x : r2.x), (uint32_t)s + 1u);               // only the positions after mine
        t1[j] = e2 ? r2.y : (e1 ? r1.y : r0.y);
    }
#pragma unroll
    for (int j = 0; j < 9; ++j) {
        for (uint32_t t = t0[j]; t < t1[j]; t += DETECT_NB) {                      // DETECT_NB candidates in flight
            uint32_t tt[DETECT_NB];
            float4 fc[DETECT_NB];
            bool nn[DETECT_NB], any = false;
#pragma unroll
            for (int b = 0; b < DETECT_NB; ++b) {
                tt[b] = min(t + (uint32_t)b, t1[j] - 1u);                          // past the end: the last candidate again
                fc[b] = xf_s[tt[b]];                                               // first look in single precision (no branch),
            }
#pragma unroll
            for (int b = 0; b < DETECT_NB; ++b) {
                nn[b] = dem_near<T, PERIODIC>(P, minef, fc[b]) & (b == 0 || tt[b] != tt[b > 0 ? b - 1 : 0]);
                any |= nn[b];
            }
            if (any) {                                                             // Eq. (2) in T for the few that pass
#pragma unroll
                for (int b = 0; b < DETECT_NB; ++b)
                    if (nn[b] && dem_touch<T, PERIODIC>(P, mine, xr_s[tt[b]])) enter(tt[b]);
            }
        }
    }
    if (PERIODIC && !P.bc[0] && (c0 == 0 || c0 == P.nc[0] - 1)) {                  // the wrapped cell of a periodic row
        const int wc = c0 == 0 ? P.nc[0] - 1 : 0;
        for (int j = 0; j < 9; ++j) {
            int qz = c2 + (j / 3 - 1), qy = c1 + (j % 3 - 1);
            if (qz < 0 || qz >= P.nc[2]) { if (P.bc[2]) continue; qz = qz < 0 ? qz + P.nc[2] : qz - P.nc[2]; }
            if (qy < 0 || qy >= P.nc[1]) { if (P.bc[1]) continue; qy = qy < 0 ? qy + P.nc[1] : qy - P.nc[1]; }
            const uint2 r = cell_range[(size_t)P.nc[0] * (size_t)(qy + P.nc[1] * qz) + wc];
            for (uint32_t t = max(r.x, (uint32_t)s + 1u); t < r.y; ++t)
                if (dem_near<T, PERIODIC>(P, minef, xf_s[t]) && dem_touch<T, PERIODIC>(P, mine, xr_s[t])) enter(t);
        }
    }
    // walls: static infinite particles; overlap decided as the oracle does, R - distance > 0
    const T xm[3] = {mine.x, mine.y, mine.z};
#pragma unroll
    for (int wl = 0; wl < 6; ++wl) {
        const int ax = wl >> 1;
        if (!P.bc[ax]) continue;
        const T dist = (wl & 1) ? P.hi[ax] - xm[ax] : xm[ax] - P.lo[ax];
        if (mine.w - dist > T(0.0)) own(DEM_WALL + (uint32_t)wl);
    }
    flush();
    return nf;
}

template <typename T, bool PERIODIC>
__global__ void __launch_bounds__(CONTACT_BLOCK, DETECT_MIN_BLOCKS) dem_detect_kernel(
    const DemDevT<T> P, const uint32_t* __restrict__ skey, const typename Real<T>::v4* __restrict__ xr_s, const float4* __restrict__ xf_s,
    const uint2* __restrict__ cell_range, uint32_t* __restrict__ nfwd, uint32_t* __restrict__ nback, uint32_t* __restrict__ cand,
    int32_t* __restrict__ status)
{
    DEM_PDL_ENTER(P.n);
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n) return;
    int st = 0;
    nfwd[s] = dem_detect_one<T, PERIODIC>(P, s, skey, xr_s, xf_s, cell_range, nback, cand, st);
    if (st) atomicOr(status, st);
}

// ------------------------------------------------------------------------------ scan
// off[s] = sum over s' < s of min(nfwd[s'] + nback[s'], maxc), off[n] = total: single pass, chained tiles with decoupled look-back
// (tiles take tickets, as in the sort).
__global__ void __launch_bounds__(SCAN_THREADS) dem_scan_kernel(int n, uint32_t maxc, const uint32_t* __restrict__ cnt,
                                                               const uint32_t* __restrict__ cnt2, uint32_t* __restrict__ off,
                                                               uint32_t* __restrict__ state, uint32_t* __restrict__ ticket)
{
    DEM_PDL_ENTER(n);
    __shared__ uint32_t sc[SCAN_SMEM];
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const long long base = (long long)tile * SCAN_TILE;
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        const int x = j * SCAN_THREADS + tid;
        sc[scan_pad(x)] = base + x < n ? min(cnt[base + x] + cnt2[base + x], maxc) : 0u;
    }
    __syncthreads();
    const uint32_t end = scan_tile_chained(sc, tile, state);
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        const int x = j * SCAN_THREADS + tid;
        if (base + x < n) off[base + x] = sc[scan_pad(x)];
    }
    if (tid == 0 && base + SCAN_TILE >= n) off[n] = end;                            // the last tile
}

// ------------------------------------------------------------------------------ fill
// One thread per particle: its list of partners, put into ascending order of the partner id (walls, id n + wall, last):
// the order of the paper's lexicographically sorted pair list, which is also the order the oracle sums
// in.  Last step's list of the particle is in the same order, so one merge finds for every end the end it continues
// (PAPER.md:496 searches the previous sorted pair list instead).  Everything the force kernel needs to start an end comes
// out as coalesced records: owner and partner (sorted position: the packed (x, R) records; home index: the predictor
// velocities) and where the previous delta_t is.
// The particle's row descriptor is renewed here; a particle that has just lost its last contact gets its sums zeroed.
#define DEM_NO_PREV 0xffffffffu
struct DemEnds { uint32_t *s, *t, *hs, *ht, *prev; };   // per contact end, CSR order

// The list of the particle at sorted position s.  tq = shared memory, uint2 [maxc][STRIDE] (partner code, partner id)
// followed by uint32 [maxc][STRIDE] (last step's partner ids); the calling thread owns column `col` of both.
template <typename T, int STRIDE>
__device__ __forceinline__ void dem_fill_one(const int n, const uint32_t maxc, const int s, const int col, uint2* tq,
                                             const uint32_t* __restrict__ nfwd, const uint32_t* __restrict__ nback,
                                             const uint32_t* __restrict__ cand, const uint32_t* __restrict__ sid,
                                             const uint32_t* __restrict__ sh, const uint32_t* __restrict__ off,
                                             uint2* __restrict__ row, T* __restrict__ fm, const uint32_t* __restrict__ hq_prev,
                                             const DemEnds& E, uint32_t* __restrict__ hq, int32_t* __restrict__ status)
{
    const uint32_t nf = min(nfwd[s], maxc), nb = min(nback[s], maxc);
    const uint32_t cnt = min(nf + nb, maxc);
    if (nf + nb > maxc) atomicOr(status, LEDDS_ST_CONTACT_OVERFLOW);                // the two ends of the column met
    const uint32_t h = sh[s];
    const uint2 old = row[h];
    if (cnt == 0) {
        if (old.y) {                                                                // the last contact has just ended
            row[h] = make_uint2(0u, 0u);
#pragma unroll
            for (int c = 0; c < 6; ++c) fm[6 * (size_t)h + c] = T(0.0);
        }
        return;
    }
    uint2* mine = tq + col;
    uint32_t* pq = reinterpret_cast<uint32_t*>(tq + (size_t)maxc * STRIDE) + col;   // last step's partner ids
    const uint32_t o = off[s];
    // every loop below keeps four independent loads in flight per thread: the partner codes, their ids, last step's
    // ids of this particle; then the ordering runs in shared memory
    for (uint32_t c0 = 0; c0 < cnt; c0 += 4) {
        uint32_t t[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t c = c0 + j;
            t[j] = c < cnt ? cand[(size_t)(c < nf ? c : maxc - 1u - (c - nf)) * n + s] : 0u;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (c0 + j < cnt) mine[(c0 + j) * STRIDE].x = t[j];
    }
    for (uint32_t c0 = 0; c0 < old.y; c0 += 4) {
        uint32_t q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = c0 + j < old.y ? hq_prev[old.x + c0 + j] : 0u;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (c0 + j < old.y) pq[(c0 + j) * STRIDE] = q[j];
    }
    for (uint32_t c0 = 0; c0 < cnt; c0 += 4) {
        uint32_t q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t t = c0 + j < cnt ? mine[(c0 + j) * STRIDE].x : DEM_WALL;
            q[j] = t >= DEM_WALL ? (uint32_t)n + (t - DEM_WALL) : sid[t];
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (c0 + j < cnt) mine[(c0 + j) * STRIDE].y = q[j];
    }
    for (uint32_t c = 1; c < cnt; ++c) {                                            // insertion sort by id
        const uint2 e = mine[c * STRIDE];
        uint32_t k = c;
        while (k > 0 && mine[(k - 1) * STRIDE].y > e.y) { mine[k * STRIDE] = mine[(k - 1) * STRIDE]; --k; }
        mine[k * STRIDE] = e;
    }
    uint32_t k = 0;
    for (uint32_t c0 = 0; c0 < cnt; c0 += 4) {
        uint2 e[4];
        uint32_t ht[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            e[j] = c0 + j < cnt ? mine[(c0 + j) * STRIDE] : make_uint2(DEM_WALL, 0u);
            ht[j] = e[j].x >= DEM_WALL ? 0u : sh[e[j].x];
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t c = c0 + j;
            if (c >= cnt) break;
            while (k < old.y && pq[k * STRIDE] < e[j].y) ++k;                 // both lists ascend in the partner id
            E.s[o + c] = (uint32_t)s;
            E.t[o + c] = e[j].x;
            E.hs[o + c] = h;
            E.ht[o + c] = ht[j];
            E.prev[o + c] = (k < old.y && pq[k * STRIDE] == e[j].y) ? old.x + k : DEM_NO_PREV;
            hq[o + c] = e[j].y;
        }
    }
    row[h] = make_uint2(o, cnt);
}

template <typename T>
__global__ void __launch_bounds__(CONTACT_BLOCK) dem_fill_kernel(int n, uint32_t maxc, const uint32_t* __restrict__ nfwd,
                                                                const uint32_t* __restrict__ nback, const uint32_t* __restrict__ cand,
                                                                const uint32_t* __restrict__ sid, const uint32_t* __restrict__ sh,
                                                                const uint32_t* __restrict__ off, uint2* __restrict__ row,
                                                                T* __restrict__ fm, const uint32_t* __restrict__ hq_prev,
                                                                const DemEnds E, uint32_t* __restrict__ hq, int32_t* __restrict__ status)
{
    DEM_PDL_ENTER(n);
    extern __shared__ uint2 tq[];                        // uint2 [maxc][CONTACT_BLOCK] + uint32 [maxc][CONTACT_BLOCK]
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    dem_fill_one<T, CONTACT_BLOCK>(n, maxc, s, (int)threadIdx.x, tq, nfwd, nback, cand, sid, sh, off, row, fm, hq_prev, E, hq, status);
}

// ------------------------------------------------------------------------------ force
// A warp owns FORCE_PW consecutive particles (sorted order) and all their contact ends, a contiguous piece
// [off[s0], off[s0 + FORCE_PW]) of the CSR arrays.  It works through that piece 32 ends at a time, one end per lane
// (all lanes busy whatever the contact counts of the particles are); the end's force and torque go to shared
// memory, and the lane that owns the particle adds up its ends in list order (Eq. 1).  An end starts from the records
// dem_fill_kernel left: one coalesced read, then every further load (both bodies, the previous delta_t) is independent
// of the others.
// Both partners evaluate their contact, each from its own side: e_n = (r_owner - r_partner)/|.|, v_rel, delta_t and the
// forces all change sign exactly when the roles are swapped (every operation below is sign-symmetric in IEEE arithmetic
// and the sums R_i w_i + R_j w_j, m_i m_j, m_i + m_j commute; no FMA contraction in this file), so F_ij = -F_ji and
// M_i / R_i = M_j / R_j hold bit for bit, and what the owner with the higher id computes is exactly the negative of the
// canonical (i < j) evaluation of the oracle.
// The FORCE_PW particles from sorted position s0 on, by one warp with its own piece of shared memory (s_off, stage, sacc).
template <typename T, bool HERTZ>
__device__ __forceinline__ void dem_force_warp(
    const DemDevT<T>& P, const int s0, const int lane, uint32_t* s_off, T (*stage)[32], T (*sacc)[FORCE_PW],
    const typename Real<T>::v4* __restrict__ xr_s, const T* __restrict__ pvw, const uint32_t* __restrict__ off,
    const DemEnds& E, const uint32_t* __restrict__ sh, T* __restrict__ fm, const T* __restrict__ hdt_prev,
    T* __restrict__ hdt_new, int32_t* __restrict__ status, const T dt_hist)
{
    const int np = min(FORCE_PW, P.n - s0);
    const uint32_t e_begin = off[s0], e_end = off[s0 + np];
    if (e_begin == e_end) return;                                                   // no contact among these particles (warp-uniform)
    for (int i = lane; i <= np; i += 32) s_off[i] = off[s0 + i];
    for (int i = lane; i < 6 * FORCE_PW; i += 32) (&sacc[0][0])[i] = T(0.0);
    __syncwarp();
    int st = 0;

    for (uint32_t chunk = e_begin; chunk < e_end; chunk += 32) {
        const uint32_t e = chunk + (uint32_t)lane;
        T Fe[3] = {0, 0, 0}, Me[3] = {0, 0, 0};
        if (e < e_end) {
            const uint32_t s = E.s[e], t = E.t[e], hs = E.hs[e], ht = E.ht[e], prev = E.prev[e];
            const bool wall = t >= DEM_WALL;
            // all loads of the end, issued together
            const typename Real<T>::v4 m4 = xr_s[s];
            const typename Real<T>::v2* rm = reinterpret_cast<const typename Real<T>::v2*>(pvw + 6 * (size_t)hs);
            const typename Real<T>::v2 ma = rm[0], mb = rm[1], mc = rm[2];
            const typename Real<T>::v4 o4 = xr_s[wall ? s : t];
            const typename Real<T>::v2* ro = reinterpret_cast<const typename Real<T>::v2*>(pvw + 6 * (size_t)(wall ? hs : ht));
            const typename Real<T>::v2 oa = ro[0], ob = ro[1], oc = ro[2];
            T dt3[3] = {0, 0, 0};                                                 // previous delta_t of this end, seen from its owner
            if (prev != DEM_NO_PREV) {
                const T* d = hdt_prev + 3 * (size_t)prev;
                dt3[0] = d[0]; dt3[1] = d[1]; dt3[2] = d[2];
            }
            const T xm[3] = {m4.x, m4.y, m4.z}, Rm = m4.w;
            const T vm[3] = {ma.x, ma.y, mb.x}, wm[3] = {mb.y, mc.x, mc.y};
            T F[3] = {0, 0, 0}, Tq[3] = {0, 0, 0}, kn, kt, gn, gt;
            if (!wall) {
                const T xo[3] = {o4.x, o4.y, o4.z}, Ro = o4.w;
                const T vo[3] = {oa.x, oa.y, ob.x}, wo[3] = {ob.y, oc.x, oc.y};
                T d[3];
                dem_min_image(P, xm, xo, d);
                const T dist = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                const T dn = (Rm + Ro) - dist;                                    // Eq. (6)
                if (dist == T(0.0)) {
                    st |= LEDDS_ST_COINCIDENT;                                         // pair skipped, delta_t = 0 (as the oracle)
                    dt3[0] = dt3[1] = dt3[2] = T(0.0);
                } else {
                    const T en[3] = {d[0] / dist, d[1] / dist, d[2] / dist};      // Eq. (7)
                    const T mi = dem_mass(P, Rm), mj = dem_mass(P, Ro);
                    const T mstar = mi * mj / (mi + mj);                          // (A.9)
                    dem_coefficients<T, HERTZ>(P.kn, P.kt, P.Ystar, P.Gstar, P.zeta, mstar, Rm * Ro / (Rm + Ro), dn, kn, kt, gn, gt);
                    dem_pair_force(en, dn, vm, wm, Rm, vo, wo, Ro, kn, kt, gn, gt, P.mu, dt_hist, dt3, F, Tq);
                }
            } else {                                                                   // a wall: R* = R_i, m* = m_i
                const int wl = (int)(t - DEM_WALL), ax = wl >> 1, side = wl & 1;
                const T xa = ax == 0 ? xm[0] : (ax == 1 ? xm[1] : xm[2]);          // selects: the arrays stay in registers
                const T dist = side ? P.hi[ax] - xa : xa - P.lo[ax];
                const T dn = Rm - dist;
                const T sgn = side ? -T(1.0) : T(1.0);
                const T en[3] = {ax == 0 ? sgn : T(0.0), ax == 1 ? sgn : T(0.0), ax == 2 ? sgn : T(0.0)};
                const T vj[3] = {P.vw[wl * 3], P.vw[wl * 3 + 1], P.vw[wl * 3 + 2]}, wj[3] = {0, 0, 0};
                dem_coefficients<T, HERTZ>(P.kn_w, P.kt_w, P.Ystar_w, P.Gstar_w, P.zeta_w, dem_mass(P, Rm), Rm, dn, kn, kt, gn, gt);
                dem_pair_force(en, dn, vm, wm, Rm, vj, wj, T(0.0), kn, kt, gn, gt, P.mu_w, dt_hist, dt3, F, Tq);
            }
#pragma unroll
            for (int a = 0; a < 3; ++a) { Fe[a] = F[a]; Me[a] = Rm * (-Tq[a]); }         // Eq. (15)
            T* nd = hdt_new + 3 * (size_t)e;
            nd[0] = dt3[0]; nd[1] = dt3[1]; nd[2] = dt3[2];
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) { stage[a][lane] = Fe[a]; stage[3 + a][lane] = Me[a]; }
        __syncwarp();
        // Eq. (1): the lane that owns a particle adds up the ends of this round that are the particle's, in list order
        for (int i = lane; i < np; i += 32) {
            const uint32_t lo = max(s_off[i], chunk), hi = min(s_off[i + 1], chunk + 32u);
            if (lo < hi) {
                T a6[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) a6[c] = sacc[c][i];
                for (uint32_t e2 = lo; e2 < hi; ++e2)
#pragma unroll
                    for (int c = 0; c < 6; ++c) a6[c] += stage[c][e2 - chunk];
#pragma unroll
                for (int c = 0; c < 6; ++c) sacc[c][i] = a6[c];
            }
        }
        __syncwarp();
    }
    // the sums of every particle that has a contact, for the kick (home order)
    for (int i = lane; i < np; i += 32) {
        if (s_off[i + 1] == s_off[i]) continue;
        const uint32_t h = sh[s0 + i];
        bool finite = true;
#pragma unroll
        for (int c = 0; c < 6; ++c) { const T v = sacc[c][i]; fm[6 * (size_t)h + c] = v; finite = finite && isfinite(v); }
        if (!finite) st |= LEDDS_ST_NONFINITE;
    }
    if (st) atomicOr(status, st);
}

template <typename T, bool HERTZ>
__global__ void __launch_bounds__(FORCE_THREADS, FORCE_MIN_BLOCKS) dem_force_kernel(
    const DemDevT<T> P, const typename Real<T>::v4* __restrict__ xr_s, const T* __restrict__ pvw, const uint32_t* __restrict__ off,
    const DemEnds E, const uint32_t* __restrict__ sh, T* __restrict__ fm, const T* __restrict__ hdt_prev,
    T* __restrict__ hdt_new, int32_t* __restrict__ status, T dt_hist)
{
    DEM_PDL_ENTER(P.n);
    // every warp works on its own FORCE_PW particles with its own piece of shared memory: no block-wide barrier
    __shared__ uint32_t s_off_all[FORCE_WARPS][FORCE_PW + 1];
    __shared__ T stage_all[FORCE_WARPS][6][32];
    __shared__ T sacc_all[FORCE_WARPS][6][FORCE_PW];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int s0 = (blockIdx.x * FORCE_WARPS + warp) * FORCE_PW;
    if (s0 >= P.n) return;
    dem_force_warp<T, HERTZ>(P, s0, lane, s_off_all[warp], stage_all[warp], sacc_all[warp], xr_s, pvw, off, E, sh, fm, hdt_prev,
                             hdt_new, status, dt_hist);
}

// ------------------------------------------------------------------------------ small systems: the step in one launch
// For a few thousand particles every kernel of the chain above runs a few microseconds and the step is bound by its
// twelve dependent launches (PAPER.md:682-712 has workloads of this size; BASELINE configs[0]: 2 048 spheres).  Here ONE
// thread-block cluster of SMALL_CTAS blocks (one per SM, 256 or 512 threads each) does the whole step -- [kick] -> drift ->
// keys -> order -> sorted copies -> detect -> scan -> fill -> force -- on the same arrays of the scratch and history
// buffers, with cluster barriers (release / acquire: ~0.2 us, the L1 caches are invalidated) where the chain has kernel
// boundaries, so import / export / query / re-homing and the coupled step see no difference.  (A single block was
// measured first: 80 us per step for 2 048 spheres, bound by what one SM can move to and from L2.)
// The order (cell key, id) is reached by a counting sort: particles count themselves into their cells (integer
// atomics), the cell counts are scanned by the cluster, and the particles of a cell are ranked by id (the ranking of
// dem_gather_kernel): a unique result, equal to that of the radix passes bit for bit.  Detection, list ordering /
// history merge and the force evaluation are the device functions of the kernels above (dem_detect_one,
// dem_fill_one, dem_force_warp), called with the cluster's threads / warps in place of a grid.
// Used when n <= SMALL_MAX_N and the grid has <= SMALL_MAX_CELLS cells (ledds_dem_params.no_single_block = 0).
#define SMALL_CTAS 8                          // portable cluster size
#define SMALL_THREADS 512                     // the most threads a block is launched with (256 for n <= 2 048: all 8 SMs busy)
#define SMALL_WARPS (SMALL_THREADS / 32)
#define SMALL_MAX_N 4096                      // measured: 1.2 x the chain of kernels at 4 096 spheres, 1.5 x at 2 048, equal at ~6 000
#define SMALL_MAX_CELLS 32768

template <typename T>
struct DemSmallArgs {
    DemDevT<T> P;
    typename Real<T>::v4* hx;                // home state
    T *hv, *hw, *ha, *hal, *pvw;
    const uint32_t* hid;
    T* fm;                                   // contact sums of the last evaluation (read by the kick, renewed by fill / force)
    uint2* row;
    const T *f_ext, *m_ext;
    uint32_t *key, *slot;                    // by home index: cell key; arrival number inside the cell
    uint32_t *htmp, *sid_tmp;                // by position before the ranking inside a cell: home index; id
    uint2* cell_range;
    uint32_t *skey, *sid, *sh;               // sorted order: key, id, home index
    typename Real<T>::v4* xr_s;
    float4* xf_s;
    uint32_t *nfwd, *nback, *cand, *off;
    uint32_t* csum;                          // 2 x SMALL_CTAS words: block totals of the two cluster-wide scans
    DemEnds E;
    const uint32_t* hq_prev;
    uint32_t* hq;
    const T* hdt_prev;
    T* hdt_new;
    int32_t* status;
    T dt_hist;
    int kick, drift;                         // kick: the first step begins with the kick of the step before the launch
    int part;                                // bit 0: kick / drift / keys / cell counts; bit 1: everything after
    int nsteps;                              // steps in this launch (> 1 only with part = 3 and drift = 1)
};

// all threads of the cluster; what they wrote before is visible to all of them after
__device__ __forceinline__ void small_sync()
{
    asm volatile("barrier.cluster.arrive.release;\n\tbarrier.cluster.wait.acquire;" ::: "memory");
}
__device__ __forceinline__ uint32_t small_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}

// exclusive prefix of v over the threads of the cluster in the order (block rank, thread), and the total.
// wsum: SMALL_WARPS words of shared memory; csum: SMALL_CTAS words of global memory, used once per launch.
__device__ __forceinline__ uint32_t small_cluster_scan(uint32_t v, uint32_t* wsum, uint32_t* csum, uint32_t rank, uint32_t& total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (int)(blockDim.x >> 5);
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();                                          // wsum may still be read from the last scan
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t before = 0, btotal = 0;
    for (int w2 = 0; w2 < nw; ++w2) {
        const uint32_t c = wsum[w2];
        if (w2 < warp) before += c;
        btotal += c;
    }
    if (threadIdx.x == 0) csum[rank] = btotal;
    small_sync();
    total = 0;
#pragma unroll
    for (uint32_t r = 0; r < SMALL_CTAS; ++r) {
        const uint32_t c = __ldcg(csum + r);
        if (r < rank) before += c;
        total += c;
    }
    return before + incl - v;
}

template <typename T, bool HERTZ, bool PERIODIC>
__global__ void __launch_bounds__(SMALL_THREADS, 1) dem_small_step_kernel(const __grid_constant__ DemSmallArgs<T> A)
{
    extern __shared__ __align__(16) unsigned char small_dyn[];
    __shared__ uint32_t wsum[SMALL_WARPS];
    const DemDevT<T>& P = A.P;
    const uint32_t rank = small_rank();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n = P.n, ncell = (int)P.ncell;
    const int nt = (int)blockDim.x, SMALL_TOTAL = SMALL_CTAS * nt, nw = nt >> 5;   // 256 or SMALL_THREADS threads per block
    const int gtid = (int)rank * nt + tid;
    const uint32_t maxc = (uint32_t)P.maxc;
    int st = 0;
    // nsteps > 1 (part = 3 only): that many steps in this one launch; the contact lists and delta_t of a step are the
    // "previous" ones of the next (the two generations change roles), and every step after the first begins with
    // the kick that closes the one before it
    const uint32_t* hq_prev = A.hq_prev;
    uint32_t* hq = A.hq;
    const T* hdt_prev = A.hdt_prev;
    T* hdt_new = A.hdt_new;
    for (int it = 0; it < A.nsteps; ++it) {
    const bool kick = it > 0 || A.kick;
    if (A.part & 1) {
        // [kick] + drift + predictor + key: the expressions of dem_drift_key_kernel, one thread per particle
        for (int h = gtid; h < n; h += SMALL_TOTAL) {
            const typename Real<T>::v4 r = A.hx[h];
            T xn[3] = {r.x, r.y, r.z};
            const T R = r.w;
            const T m = dem_mass(P, R), I = T(0.4) * m * R * R;               // Eq. (21a)
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const size_t e = 3 * (size_t)h + k;
                T vv = A.hv[e], wv = A.hw[e], av = A.ha[e], alv = A.hal[e];
                if (kick) {
                    const size_t ie = (A.f_ext || A.m_ext) ? 3 * (size_t)A.hid[h] + k : 0;
                    const T Fq = A.fm[6 * (size_t)h + k] + (A.f_ext ? A.f_ext[ie] : T(0.0)), Mq = A.fm[6 * (size_t)h + 3 + k] + (A.m_ext ? A.m_ext[ie] : T(0.0));
                    const T an = dem_div0(Fq, m) + P.g[k], aln = dem_div0(Mq, I);                  // Eq. (18b), (19c)
                    vv = vv + (T(0.5) * P.dt) * (av + an);                               // Eq. (18c)
                    wv = wv + (T(0.5) * P.dt) * (alv + aln);                             // Eq. (19d)
                    av = an; alv = aln;
                    A.hv[e] = vv; A.hw[e] = wv; A.ha[e] = av; A.hal[e] = alv;
                }
                if (A.drift) {
                    A.pvw[6 * (size_t)h + k] = vv + (T(0.5) * P.dt) * av;                // predictor (G11)
                    A.pvw[6 * (size_t)h + 3 + k] = wv + (T(0.5) * P.dt) * alv;
                    T xv = xn[k] + P.dt * vv + (T(0.5) * P.dt * P.dt) * av;              // Eq. (18a)
                    if (!P.bc[k]) {
                        if (xv >= P.hi[k]) xv -= P.L[k];
                        else if (xv < P.lo[k]) xv += P.L[k];
                    }
                    xn[k] = xv;
                } else {
                    A.pvw[6 * (size_t)h + k] = vv;
                    A.pvw[6 * (size_t)h + 3 + k] = wv;
                }
            }
            if (A.drift) A.hx[h] = Real<T>::make4(xn[0], xn[1], xn[2], r.w);
            const int cx = dem_cell_coord(P, xn[0], 0), cy = dem_cell_coord(P, xn[1], 1), cz = dem_cell_coord(P, xn[2], 2);
            const uint32_t key = (uint32_t)(cx + P.nc[0] * (cy + P.nc[1] * cz));
            A.key[h] = key;
            A.slot[h] = atomicAdd(&A.cell_range[key].y, 1u);                  // the particle's number among those of its cell
            if (T(2.0) * r.w > P.hmin) st |= LEDDS_ST_RADIUS_RANGE;          // input contract (include/ledds.h)
#pragma unroll
            for (int a = 0; a < 3; ++a)
                if (P.bc[a] && !(xn[a] >= P.lo[a] && xn[a] <= P.hi[a])) st |= LEDDS_ST_OUT_OF_BOX;
        }
    }
    if (A.part == 3) small_sync();
    if (A.part & 2) {
        // cell counts -> [start, end): every thread sums a contiguous piece of the cells, the cluster scans the sums.
        // The counts were made by atomics (in L2): they are read past the L1 cache.
        {
            const int per = (ncell + SMALL_TOTAL - 1) / SMALL_TOTAL;
            const int c0 = min(ncell, gtid * per), c1 = min(ncell, c0 + per);
            uint32_t sum = 0;
            for (int c = c0; c < c1; ++c) sum += __ldcg(&A.cell_range[c].y);
            uint32_t total;
            uint32_t run = small_cluster_scan(sum, wsum, A.csum, rank, total);
            for (int c = c0; c < c1; ++c) {
                const uint32_t k = __ldcg(&A.cell_range[c].y);
                if (k) A.cell_range[c] = make_uint2(run, run + k);
                run += k;
            }
        }
        small_sync();
        for (int h = gtid; h < n; h += SMALL_TOTAL) {                         // into the cell, in arrival order
            const uint32_t p = A.cell_range[A.key[h]].x + A.slot[h];
            A.sid_tmp[p] = A.hid[h];
            A.htmp[p] = (uint32_t)h;
        }
        small_sync();
        for (int p = gtid; p < n; p += SMALL_TOTAL) {                         // rank by id inside the cell, sorted copies
            const uint32_t h = A.htmp[p], key = A.key[h], id = A.sid_tmp[p];
            const uint2 cr = A.cell_range[key];
            uint32_t s = cr.x;
            for (uint32_t t = cr.x; t < cr.y; ++t) s += A.sid_tmp[t] < id;   // ids are distinct
            A.skey[s] = key;
            const typename Real<T>::v4 r = A.hx[h];
            A.xr_s[s] = r;
            A.sid[s] = id;
            A.sh[s] = h;
            A.nback[s] = 0u;
            const T rx = r.x - P.lo[0], ry = r.y - P.lo[1], rz = r.z - P.lo[2];   // as dem_gather_kernel
            const bool sane = fabs(rx) <= T(2.0) * P.L[0] && fabs(ry) <= T(2.0) * P.L[1] && fabs(rz) <= T(2.0) * P.L[2];
            const float qnan = __int_as_float(0x7fc00000);
            A.xf_s[s] = sane ? make_float4((float)rx, (float)ry, (float)rz, (float)r.w) : make_float4(qnan, qnan, qnan, qnan);
        }
        small_sync();
        for (int s = gtid; s < n; s += SMALL_TOTAL)
            A.nfwd[s] = dem_detect_one<T, PERIODIC>(P, s, A.skey, A.xr_s, A.xf_s, A.cell_range, A.nback, A.cand, st);
        small_sync();
        // the cell ranges have done their work: all cells empty again for the next step's counts (the first step of a
        // handle finds them cleared by the host)
        for (int c = gtid; c < ncell; c += SMALL_TOTAL) A.cell_range[c] = make_uint2(0u, 0u);
        {   // off[s] = sum over s' < s of min(nfwd + nback, maxc), off[n] = total (nback was counted by atomics)
            const int per = (n + SMALL_TOTAL - 1) / SMALL_TOTAL;
            const int i0 = min(n, gtid * per), i1 = min(n, i0 + per);
            uint32_t sum = 0;
            for (int i = i0; i < i1; ++i) sum += min(A.nfwd[i] + __ldcg(A.nback + i), maxc);
            uint32_t total;
            uint32_t run = small_cluster_scan(sum, wsum, A.csum + SMALL_CTAS, rank, total);
            for (int i = i0; i < i1; ++i) {
                A.off[i] = run;
                run += min(A.nfwd[i] + __ldcg(A.nback + i), maxc);
            }
            if (gtid == 0) A.off[n] = total;
        }
        small_sync();
        {
            uint2* tq = reinterpret_cast<uint2*>(small_dyn);
            for (int s = gtid; s < n; s += SMALL_TOTAL)
                dem_fill_one<T, SMALL_THREADS>(n, maxc, s, tid, tq, A.nfwd, A.nback, A.cand, A.sid, A.sh, A.off, A.row, A.fm,
                                               hq_prev, A.E, hq, A.status);
        }
        small_sync();
        {   // a warp's piece of shared memory: s_off (FORCE_PW + 1 words, padded), stage [6][32], sacc [6][FORCE_PW]
            constexpr size_t per_warp = 272 + (6 * 32 + 6 * FORCE_PW) * sizeof(T);
            unsigned char* mine = small_dyn + (size_t)warp * per_warp;
            uint32_t* s_off = reinterpret_cast<uint32_t*>(mine);
            T (*stage)[32] = reinterpret_cast<T (*)[32]>(mine + 272);
            T (*sacc)[FORCE_PW] = reinterpret_cast<T (*)[FORCE_PW]>(mine + 272 + 6 * 32 * sizeof(T));
            for (int s0 = ((int)rank * nw + warp) * FORCE_PW; s0 < n; s0 += SMALL_CTAS * nw * FORCE_PW) {
                dem_force_warp<T, HERTZ>(P, s0, lane, s_off, stage, sacc, A.xr_s, A.pvw, A.off, A.E, A.sh, A.fm, hdt_prev,
                                         hdt_new, A.status, A.dt_hist);
                __syncwarp();
            }
        }
    }
    if (it + 1 < A.nsteps) {
        small_sync();                                          // the sums and lists of this step before the next one's kick
        const uint32_t* q = hq_prev; hq_prev = hq; hq = const_cast<uint32_t*>(q);
        const T* d = hdt_prev; hdt_prev = hdt_new; hdt_new = const_cast<T*>(d);
    }
    }
    if (st) atomicOr(A.status, st);
}

// shared memory a block is launched with: the larger of the fill phase's and the force phase's needs
template <typename T>
static size_t dem_small_smem(int maxc)
{
    const size_t fill = (size_t)maxc * SMALL_THREADS * 12, force = (size_t)SMALL_WARPS * (272 + (6 * 32 + 6 * FORCE_PW) * sizeof(T));
    return fill > force ? fill : force;
}

// ------------------------------------------------------------------------------ kick
// One thread per vector component (element e = 3 h + k of the flat home arrays): coalesced.
template <typename T>
__global__ void dem_kick_kernel(const DemDevT<T> P, const typename Real<T>::v4* __restrict__ hx, const uint32_t* __restrict__ hid,
                                const T* __restrict__ fm, const T* __restrict__ f_ext, const T* __restrict__ m_ext,
                                T* __restrict__ hv, T* __restrict__ hw, T* __restrict__ ha, T* __restrict__ hal,
                                int only_accel)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= 3ll * P.n) return;
    const int h = (int)(e / 3), k = (int)(e - 3ll * h);
    const T R = reinterpret_cast<const T*>(hx)[4 * (size_t)h + 3];
    const T m = dem_mass(P, R), I = T(0.4) * m * R * R;                             // Eq. (21a)
    const size_t ie = (f_ext || m_ext) ? 3 * (size_t)hid[h] + k : 0;
    const T Fq = fm[6 * (size_t)h + k] + (f_ext ? f_ext[ie] : T(0.0)), Mq = fm[6 * (size_t)h + 3 + k] + (m_ext ? m_ext[ie] : T(0.0));
    const T an = Fq / m + P.g[k], aln = Mq / I;                                  // Eq. (18b), (19c)
    if (!only_accel) {
        hv[e] = hv[e] + (T(0.5) * P.dt) * (ha[e] + an);                                  // Eq. (18c)
        hw[e] = hw[e] + (T(0.5) * P.dt) * (hal[e] + aln);                                // Eq. (19d)
    }
    ha[e] = an;
    hal[e] = aln;
}

// ------------------------------------------------------------------------------ query (parity only)
__global__ void dem_query_pos_kernel(int n, const uint32_t* __restrict__ sid, uint32_t* __restrict__ pos_of_id)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) pos_of_id[sid[s]] = (uint32_t)s;
}

// contact ends of particle id p with a partner of higher id: the pairs (p, q) of the canonical list
__global__ void dem_pair_count_kernel(int n, const uint32_t* __restrict__ pos_of_id, const uint32_t* __restrict__ off,
                                      const uint32_t* __restrict__ hq, uint32_t* __restrict__ cnt)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const uint32_t s = pos_of_id[p];
    uint32_t c = 0;
    for (uint32_t e = off[s]; e < off[s + 1]; ++e) c += hq[e] > (uint32_t)p;
    cnt[p] = c;
}

template <typename T>
__global__ void dem_unpack_fm_kernel(int n, const uint32_t* __restrict__ hid, const T* __restrict__ fm,
                                     T* __restrict__ force, T* __restrict__ torque)
{
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n) return;
    const size_t p = hid[h];
    for (int a = 0; a < 3; ++a) {
        if (force) force[3 * p + a] = fm[6 * (size_t)h + a];
        if (torque) torque[3 * p + a] = fm[6 * (size_t)h + 3 + a];
    }
}

// single-block exclusive scan of cnt[n] into off[n+1]
__global__ void __launch_bounds__(1024) dem_block_scan_kernel(int n, const uint32_t* __restrict__ cnt, uint32_t* __restrict__ off)
{
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + tid;
        const uint32_t c = i < n ? cnt[i] : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t s = wsum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, s, o);
                if (lane >= o) s += t;
            }
            wsum[lane] = s;
        }
        __syncthreads();
        const uint32_t before = carry + (warp ? wsum[warp - 1] : 0u) + incl - c;
        if (i < n) off[i] = before;
        __syncthreads();
        if (tid == 1023) carry = before + c;
        __syncthreads();
    }
    if (tid == 0) off[n] = carry;
}

// the list of a particle is in ascending order of the partner id already (dem_fill_kernel)
template <typename T>
__global__ void dem_pair_write_kernel(int n, const uint32_t* __restrict__ pos_of_id, const uint32_t* __restrict__ off,
                                      const uint32_t* __restrict__ hq, const T* __restrict__ hdt,
                                      const uint32_t* __restrict__ pair_off, uint32_t cap, uint32_t* __restrict__ pairs,
                                      T* __restrict__ pair_dt, uint32_t* __restrict__ n_pairs)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p == 0 && n_pairs) *n_pairs = pair_off[n];
    if (p >= n) return;
    const uint32_t s = pos_of_id[p];
    uint32_t o = pair_off[p];
    for (uint32_t e = off[s]; e < off[s + 1]; ++e) {
        const uint32_t q = hq[e];
        if (q <= (uint32_t)p) continue;
        if (o >= cap) break;
        if (pairs) { pairs[2 * (size_t)o] = (uint32_t)p; pairs[2 * (size_t)o + 1] = q; }
        if (pair_dt)
            for (int a = 0; a < 3; ++a) pair_dt[3 * (size_t)o + a] = hdt[3 * (size_t)e + a];
        ++o;
    }
}

// ------------------------------------------------------------------------------ host API
static double dem_zeta_host(double eps)
{
    if (eps >= 1.0) return 0.0;
    const double l = log(eps);
    return -l / sqrt(l * l + DEM_PI * DEM_PI);                                        // -beta of (A.5)
}

// es = bytes of the handle's real type (8: fp64 calls, 4: the _f32 calls)
static int dem_setup(const ledds_dem_params* p, ledds_dem* h, size_t es)
{
    if (!p || p->n < 0 || p->max_contacts < 1 || p->max_contacts > 32) return LEDDS_EINVAL;   // n = 0: a valid, empty system
    if (!(p->cell > 0.0) || !(p->dt >= 0.0) || !(p->density > 0.0)) return LEDDS_EINVAL;
    if (p->model == 0 && (!(p->kn > 0.0) || !(p->kt > 0.0) || !(p->kn_w > 0.0) || !(p->kt_w > 0.0))) return LEDDS_EINVAL;
    if (!(p->restitution > 0.0) || !(p->restitution_w > 0.0) || p->mu < 0.0 || p->mu_w < 0.0) return LEDDS_EINVAL;
    if ((unsigned long long)p->n * (unsigned long long)p->max_contacts >= (1ull << 30)) return LEDDS_EINVAL;   // scan descriptors: 30 bits
    h->p = *p;
    DemDev& d = h->d;
    d.n = p->n;
    double ncell = 1.0;
    d.hmin = 1.0e300;
    for (int a = 0; a < 3; ++a) {
        if (!(p->hi[a] > p->lo[a]) || (p->bc[a] != 0 && p->bc[a] != 1)) return LEDDS_EINVAL;
        d.lo[a] = p->lo[a]; d.hi[a] = p->hi[a]; d.L[a] = p->hi[a] - p->lo[a]; d.bc[a] = p->bc[a];
        d.Lf[a] = (float)d.L[a];
        int nc = (int)floor(d.L[a] / p->cell);
        if (nc < 1) nc = 1;
        if (!p->bc[a] && nc < 3) return LEDDS_EINVAL;          // a periodic axis needs >= 3 cells (27-cell walk)
        d.nc[a] = nc;
        d.inv_h[a] = (double)nc / d.L[a];
        d.hmin = fmin(d.hmin, d.L[a] / (double)nc);
        d.g[a] = p->g[a];
        ncell *= nc;
        for (int s = 0; s < 2; ++s)
            for (int c = 0; c < 3; ++c) d.vw[(a * 2 + s) * 3 + c] = p->v_wall[a][s][c];
    }
    if (ncell > 4.0e9) return LEDDS_EINVAL;
    d.ncell = (unsigned)ncell;
    d.plane = (unsigned)d.nc[0] * (unsigned)d.nc[1];
    // floor(k m / 2^40) = floor(k / d) for m = ceil(2^40 / d) whenever k (m d - 2^40) < 2^40, which k d <= 2^40 ensures
    d.magic_ok = ncell * (double)d.plane <= 1099511627776.0 && (double)d.plane * d.nc[0] <= 1099511627776.0;
    d.magic_row = ((1ull << 40) + (unsigned)d.nc[0] - 1) / (unsigned)d.nc[0];
    d.magic_plane = ((1ull << 40) + d.plane - 1) / d.plane;
    d.fmargin = (float)(fmax(d.L[0], fmax(d.L[1], d.L[2])) / 524288.0);              // 2^-19 max L (dem_near)
    d.dt = p->dt; d.density = p->density;
    d.kn = p->kn; d.kt = p->kt; d.zeta = dem_zeta_host(p->restitution); d.mu = p->mu;
    d.kn_w = p->kn_w; d.kt_w = p->kt_w; d.zeta_w = dem_zeta_host(p->restitution_w); d.mu_w = p->mu_w;
    d.maxc = p->max_contacts;
    d.Ystar = d.Gstar = d.Ystar_w = d.Gstar_w = 0.0;
    if (p->model != 0 && p->model != 1) return LEDDS_EINVAL;
    if (p->model == 1) {                                                              // (A.6), (A.7)
        const double Ei = p->young, ni = p->poisson, Ew = p->young_w, nw = p->poisson_w;
        if (!(Ei > 0.0) || !(Ew > 0.0) || !(ni > -1.0 && ni < 0.5 + 1e-12) || !(nw > -1.0 && nw < 0.5 + 1e-12)) return LEDDS_EINVAL;
        d.Ystar = 1.0 / ((1.0 - ni * ni) / Ei + (1.0 - ni * ni) / Ei);
        d.Gstar = 1.0 / (2.0 * (2.0 - ni) * (1.0 + ni) / Ei + 2.0 * (2.0 - ni) * (1.0 + ni) / Ei);
        d.Ystar_w = 1.0 / ((1.0 - ni * ni) / Ei + (1.0 - nw * nw) / Ew);
        d.Gstar_w = 1.0 / (2.0 * (2.0 - ni) * (1.0 + ni) / Ei + 2.0 * (2.0 - nw) * (1.0 + nw) / Ew);
    }
    int bits = 1;
    while (bits < 32 && (1ull << bits) < (unsigned long long)d.ncell) ++bits;
    h->key_bits = bits;
    h->passes = (bits + 7) / 8;
    h->tiles = (p->n + SORT_TILE - 1) / SORT_TILE;
    h->scan_tiles = (p->n + SCAN_TILE - 1) / SCAN_TILE;
    h->cell_tiles = (int)((d.ncell + SCAN_TILE - 1) / SCAN_TILE);
    if (p->cell_order < 0 || p->cell_order > 2) return LEDDS_EINVAL;
    h->counting = p->cell_order == 2 || (p->cell_order == 0 && (double)d.ncell <= 4.0 * (double)p->n);

    const size_t n = (size_t)p->n, ecap = n * (size_t)d.maxc;
    size_t o = 0;
    DemScratch& s = h->s;
    auto take = [&](size_t bytes) { const size_t at = o; o += align_up(bytes); return at; };
    // zeroed before every step: histograms, tickets, look-back descriptors, cell ranges (kept contiguous)
    s.hist_digit = take(4 * SORT_RADIX * 4);
    s.tile_counter = take(8 * 4);
    s.tile_state = take((size_t)4 * h->tiles * SORT_RADIX * 4);
    s.scan_state = take(((size_t)h->scan_tiles + 1) * 4);
    s.cell_scan_state = take(((size_t)h->cell_tiles + 1) * 4);
    s.cell_range = take((size_t)d.ncell * 8);
    for (int b = 0; b < 2; ++b) { s.key[b] = take(n * 4); s.idx[b] = take(n * 4); }
    s.hid = take(n * 4); s.sid = take(n * 4); s.sid_tmp = take(n * 4); s.skey_f = take(n * 4);
    s.hx = take(n * 4 * es);
    s.hv = take(n * 3 * es); s.hw = take(n * 3 * es); s.ha = take(n * 3 * es); s.hal = take(n * 3 * es);
    s.pvw = take(n * 6 * es);
    s.xr_s = take(n * 4 * es); s.xf_s = take(n * 16);
    s.nfwd = take(n * 4); s.nback = take(n * 4); s.cand = take(ecap * 4);
    s.off = take((n + 1) * 4);
    s.end_s = take(ecap * 4); s.end_t = take(ecap * 4); s.end_hs = take(ecap * 4); s.end_ht = take(ecap * 4); s.end_prev = take(ecap * 4);
    s.pair_count = take((n + 1) * 4); s.pair_off = take((n + 1) * 4); s.pos_of_id = take((n + 1) * 4);
    s.total = o;

    DemHistory& hs = h->hs;
    o = 0;
    for (int b = 0; b < 2; ++b) {
        hs.fm[b] = take(n * 6 * es);
        hs.row[b] = take(n * 8);
        hs.hq[b] = take(ecap * 4);
        hs.hdt[b] = take(ecap * 3 * es);
    }
    hs.total = o;
    h->f32 = es == 4;
    {   // the same parameters in float for the kernels of an fp32 handle
        DemDevT<float>& f = h->df;
        f.n = d.n; f.fmargin = d.fmargin; f.ncell = d.ncell; f.plane = d.plane; f.magic_row = d.magic_row;
        f.magic_plane = d.magic_plane; f.magic_ok = d.magic_ok; f.hmin = (float)d.hmin; f.dt = (float)d.dt;
        f.density = (float)d.density; f.maxc = d.maxc;
        f.kn = (float)d.kn; f.kt = (float)d.kt; f.zeta = (float)d.zeta; f.mu = (float)d.mu;
        f.kn_w = (float)d.kn_w; f.kt_w = (float)d.kt_w; f.zeta_w = (float)d.zeta_w; f.mu_w = (float)d.mu_w;
        f.Ystar = (float)d.Ystar; f.Gstar = (float)d.Gstar; f.Ystar_w = (float)d.Ystar_w; f.Gstar_w = (float)d.Gstar_w;
        for (int a = 0; a < 3; ++a) {
            f.lo[a] = (float)d.lo[a]; f.hi[a] = (float)d.hi[a]; f.L[a] = (float)d.L[a]; f.Lf[a] = d.Lf[a]; f.bc[a] = d.bc[a];
            f.nc[a] = d.nc[a]; f.inv_h[a] = (float)d.inv_h[a]; f.g[a] = (float)d.g[a];
        }
        for (int k = 0; k < 18; ++k) f.vw[k] = (float)d.vw[k];
    }
    h->cur = 0;
    h->rec = 0;
    h->sorted_buf = 0;
    h->sh_buf = 0;
    h->have_sort = false;
    h->steps = 0;
    h->small_cells_clear = false;
    return LEDDS_OK;
}

static int dem_workspace_bytes(const ledds_dem_params* p, size_t* scratch_bytes, size_t* history_bytes, size_t es)
{
    ledds_dem tmp;
    const int rc = dem_setup(p, &tmp, es);
    if (rc) return rc;
    if (scratch_bytes) *scratch_bytes = tmp.s.total;
    if (history_bytes) *history_bytes = tmp.hs.total;
    return LEDDS_OK;
}
extern "C" int ledds_dem_workspace_bytes(const ledds_dem_params* p, size_t* scratch_bytes, size_t* history_bytes)
{
    return dem_workspace_bytes(p, scratch_bytes, history_bytes, 8);
}
extern "C" int ledds_dem_workspace_bytes_f32(const ledds_dem_params* p, size_t* scratch_bytes, size_t* history_bytes)
{
    return dem_workspace_bytes(p, scratch_bytes, history_bytes, 4);
}

// the kernel-side parameters of a handle in the real type T
template <typename T> static const DemDevT<T>& dem_dev(const ledds_dem* h);
template <> const DemDevT<double>& dem_dev<double>(const ledds_dem* h) { return h->d; }
template <> const DemDevT<float>& dem_dev<float>(const ledds_dem* h) { return h->df; }

template <typename T>
static T* at(void* base, size_t off) { return reinterpret_cast<T*>(static_cast<char*>(base) + off); }
template <typename T>
static const T* at(const void* base, size_t off) { return reinterpret_cast<const T*>(static_cast<const char*>(base) + off); }

// The caller's arrays in the home order of this call: the sorted order of the last sort (identity before the first).
template <typename T>
static int dem_import_t(ledds_dem* h, const T* x, const T* v, const T* w, const T* a, const T* alpha,
                     const T* radius, void* history, void* scratch, cudaStream_t st)
{
    const int n = h->d.n;
    if (n == 0) return LEDDS_OK;
    const DemScratch& s = h->s;
    const DemHistory& hs = h->hs;
    const int from = h->rec, to = 1 - h->rec;
    const uint32_t* hid_src = h->have_sort ? at<uint32_t>(scratch, s.sid) : nullptr;
    const uint32_t* perm = h->have_sort ? at<uint32_t>(scratch, s.idx[h->sh_buf]) : nullptr;
    dem_import_kernel<T><<<(n + DRIFT_BLOCK - 1) / DRIFT_BLOCK, DRIFT_BLOCK, 0, st>>>(
        n, hid_src, perm, x, v, w, a, alpha, radius, at<uint32_t>(scratch, s.hid), at<typename Real<T>::v4>(scratch, s.hx),
        at<T>(scratch, s.hv), at<T>(scratch, s.hw), at<T>(scratch, s.ha), at<T>(scratch, s.hal),
        at<T>(history, hs.fm[from]), at<uint2>(history, hs.row[from]), at<T>(history, hs.fm[to]),
        at<uint2>(history, hs.row[to]));
    LEDDS_CHECK_LAUNCH();
    h->rec = to;
    h->have_sort = false;                                      // idx[] no longer maps sorted positions to this home order
    return LEDDS_OK;
}

template <typename T>
static int dem_export_t(ledds_dem* h, T* x, T* v, T* w, T* a, T* alpha, const void* scratch, cudaStream_t st)
{
    const int n = h->d.n;
    if (n == 0) return LEDDS_OK;
    const DemScratch& s = h->s;
    dem_export_kernel<T><<<(n + DRIFT_BLOCK - 1) / DRIFT_BLOCK, DRIFT_BLOCK, 0, st>>>(
        n, at<uint32_t>(scratch, s.hid), at<typename Real<T>::v4>(scratch, s.hx), at<T>(scratch, s.hv), at<T>(scratch, s.hw),
        at<T>(scratch, s.ha), at<T>(scratch, s.hal), x, v, w, a, alpha);
    LEDDS_CHECK_LAUNCH();
    return LEDDS_OK;
}

// The single-block step (dem_small_step_kernel) in place of the chain of launches below.
static bool dem_small_ok(const ledds_dem* h)
{
    return !h->p.no_single_block && h->d.n <= SMALL_MAX_N && h->d.ncell <= SMALL_MAX_CELLS;
}

template <typename T, bool HERTZ, bool PERIODIC>
static int dem_small_launch(const DemSmallArgs<T>& A, cudaStream_t st)
{
    static bool sized[64];                                     // per device: the opt-in to > 48 KB of dynamic shared memory
    const size_t smem = dem_small_smem<T>(A.P.maxc);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return LEDDS_ECUDA;
    if (dev < 0 || dev >= 64 || !sized[dev]) {
        if (cudaFuncSetAttribute(dem_small_step_kernel<T, HERTZ, PERIODIC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)dem_small_smem<T>(32)) != cudaSuccess)
            return LEDDS_ECUDA;
        if (dev >= 0 && dev < 64) sized[dev] = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(SMALL_CTAS); cfg.blockDim = dim3(A.P.n <= SMALL_CTAS * 256 ? 256 : SMALL_THREADS); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = SMALL_CTAS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, dem_small_step_kernel<T, HERTZ, PERIODIC>, A) != cudaSuccess) return LEDDS_ECUDA;
    LEDDS_CHECK_LAUNCH();
    return LEDDS_OK;
}

// nsteps > 1: that many steps in one launch (no fork); ext = the external force / torque of every kick after the first
template <typename T>
static int dem_small_advance(ledds_dem* h, void* history, void* scratch, int32_t* status, double dt_hist, bool drift,
                             cudaStream_t st, bool fork, const DemKickT<T>* kick, int nsteps = 1,
                             const DemKickT<T>* ext = nullptr)
{
    if (nsteps > 1 && (fork || !drift)) return LEDDS_EINVAL;
    if (!ext) ext = kick;
    const DemScratch& s = h->s;
    const DemHistory& hs = h->hs;
    const int prev = h->cur, nw = 1 - h->cur;
    DemSmallArgs<T> A;
    A.P = dem_dev<T>(h);
    A.hx = at<typename Real<T>::v4>(scratch, s.hx);
    A.hv = at<T>(scratch, s.hv); A.hw = at<T>(scratch, s.hw); A.ha = at<T>(scratch, s.ha); A.hal = at<T>(scratch, s.hal);
    A.pvw = at<T>(scratch, s.pvw);
    A.hid = at<uint32_t>(scratch, s.hid);
    A.fm = at<T>(history, hs.fm[h->rec]);
    A.row = at<uint2>(history, hs.row[h->rec]);
    A.f_ext = ext ? ext->f_ext : nullptr;
    A.m_ext = ext ? ext->m_ext : nullptr;
    A.nsteps = nsteps;
    A.key = at<uint32_t>(scratch, s.key[0]); A.slot = at<uint32_t>(scratch, s.idx[0]);
    A.htmp = at<uint32_t>(scratch, s.key[1]); A.sid_tmp = at<uint32_t>(scratch, s.sid_tmp);
    A.cell_range = at<uint2>(scratch, s.cell_range);
    A.skey = at<uint32_t>(scratch, s.skey_f); A.sid = at<uint32_t>(scratch, s.sid); A.sh = at<uint32_t>(scratch, s.idx[1]);
    A.xr_s = at<typename Real<T>::v4>(scratch, s.xr_s);
    A.xf_s = at<float4>(scratch, s.xf_s);
    A.nfwd = at<uint32_t>(scratch, s.nfwd); A.nback = at<uint32_t>(scratch, s.nback);
    A.cand = at<uint32_t>(scratch, s.cand); A.off = at<uint32_t>(scratch, s.off);
    A.csum = at<uint32_t>(scratch, s.hist_digit);            // the radix histograms are not used on this path
    A.E = {at<uint32_t>(scratch, s.end_s), at<uint32_t>(scratch, s.end_t), at<uint32_t>(scratch, s.end_hs),
           at<uint32_t>(scratch, s.end_ht), at<uint32_t>(scratch, s.end_prev)};
    A.hq_prev = at<uint32_t>(history, hs.hq[prev]); A.hq = at<uint32_t>(history, hs.hq[nw]);
    A.hdt_prev = at<T>(history, hs.hdt[prev]); A.hdt_new = at<T>(history, hs.hdt[nw]);
    A.status = status;
    A.dt_hist = (T)dt_hist;
    A.kick = kick ? 1 : 0;
    A.drift = drift ? 1 : 0;
    const bool hertz = h->p.model == 1, periodic = !(A.P.bc[0] && A.P.bc[1] && A.P.bc[2]);
    auto launch = [&](int part, cudaStream_t on) {
        A.part = part;
        if (hertz) return periodic ? dem_small_launch<T, true, true>(A, on) : dem_small_launch<T, true, false>(A, on);
        return periodic ? dem_small_launch<T, false, true>(A, on) : dem_small_launch<T, false, false>(A, on);
    };
    if (!h->small_cells_clear) {
        if (cudaMemsetAsync(A.cell_range, 0, (size_t)A.P.ncell * sizeof(uint2), st) != cudaSuccess) return LEDDS_ECUDA;
        h->small_cells_clear = true;
    }
    int rc;
    if (!fork) {
        ledds_prof_start(LEDDS_K_DEM_CONTACT, st);
        rc = launch(3, st);
        ledds_prof_stop(LEDDS_K_DEM_CONTACT, st);
        if (rc) return rc;
    } else {
        // drift and keys on the caller's stream (the raster of a coupled step needs the new positions), the rest beside it
        ledds_prof_start(LEDDS_K_DEM_KEYS, st);
        rc = launch(1, st);
        ledds_prof_stop(LEDDS_K_DEM_KEYS, st);
        if (rc) return rc;
        if (!h->side && (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
                         cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                         cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess))
            return LEDDS_ECUDA;
        if (cudaEventRecord(h->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(h->side, h->ev_fork, 0) != cudaSuccess)
            return LEDDS_ECUDA;
        ledds_prof_start(LEDDS_K_DEM_CONTACT, h->side);
        rc = launch(2, h->side);
        ledds_prof_stop(LEDDS_K_DEM_CONTACT, h->side);
        if (rc) return rc;
        if (cudaEventRecord(h->ev_join, h->side) != cudaSuccess) return LEDDS_ECUDA;
    }
    h->sorted_buf = 1;
    h->sh_buf = 1;                                             // idx[1] = home index of every sorted position
    h->have_sort = true;
    h->cur = (nsteps & 1) ? nw : prev;
    return LEDDS_OK;
}

// [kick] -> drift (optional) -> keys -> sort -> gather/ranges -> contacts, all on the home state.  Leaves the contact
// sums of every particle in history (fm, row) and the contact ends in hq / hdt of the new generation.
template <typename T>
static int dem_advance_t(ledds_dem* h, void* history, void* scratch, int32_t* status, double dt_hist,
                               bool drift, cudaStream_t st, bool fork, const DemKickT<T>* kick)
{
    // kick != nullptr: the kick that closes the previous step (with the contact sums still in fm and the
    // external force / torque of *kick) is fused into the drift kernel of this one.
    // fork = true: everything after the drift/key kernel is enqueued on the handle's side stream (ordered after
    // that kernel by an event); the caller joins by waiting on h->ev_join before it needs the contact forces.
    const DemDevT<T>& d = dem_dev<T>(h);
    const DemScratch& s = h->s;
    const DemHistory& hs = h->hs;
    const int n = d.n, tb = 128, nb = (n + tb - 1) / tb;
    if (n == 0) { h->cur = 1 - h->cur; return LEDDS_OK; }
    if (dem_small_ok(h)) return dem_small_advance<T>(h, history, scratch, status, dt_hist, drift, st, fork, kick);
    g_pdl = n <= DEM_PDL_MAX_N;
    // clear sort / scan bookkeeping + cell ranges (one contiguous region)
    if (cudaMemsetAsync(at<char>(scratch, s.hist_digit), 0, s.key[0] - s.hist_digit, st) != cudaSuccess) return LEDDS_ECUDA;
    T* fm = at<T>(history, hs.fm[h->rec]);
    uint2* row = at<uint2>(history, hs.row[h->rec]);
    uint2* const cells = h->counting ? at<uint2>(scratch, s.cell_range) : nullptr;
    ledds_prof_start(LEDDS_K_DEM_KEYS, st);
    {
        const dim3 grid((n + DRIFT_BLOCK - 1) / DRIFT_BLOCK);
        if (kick)
            dem_drift_key_kernel<T, true><<<grid, DRIFT_BLOCK, 0, st>>>(d, at<typename Real<T>::v4>(scratch, s.hx), at<T>(scratch, s.hv), at<T>(scratch, s.hw),
                                                                      at<T>(scratch, s.ha), at<T>(scratch, s.hal), at<uint32_t>(scratch, s.hid), fm,
                                                                      kick->f_ext, kick->m_ext, at<T>(scratch, s.pvw),
                                                                      at<uint32_t>(scratch, s.key[0]), at<uint32_t>(scratch, s.idx[0]), drift ? 1 : 0, status, cells);
        else
            dem_drift_key_kernel<T, false><<<grid, DRIFT_BLOCK, 0, st>>>(d, at<typename Real<T>::v4>(scratch, s.hx), at<T>(scratch, s.hv), at<T>(scratch, s.hw),
                                                                       at<T>(scratch, s.ha), at<T>(scratch, s.hal), at<uint32_t>(scratch, s.hid), fm,
                                                                       nullptr, nullptr, at<T>(scratch, s.pvw),
                                                                       at<uint32_t>(scratch, s.key[0]), at<uint32_t>(scratch, s.idx[0]), drift ? 1 : 0, status, cells);
    }
    ledds_prof_stop(LEDDS_K_DEM_KEYS, st);
    LEDDS_CHECK_LAUNCH();
    if (fork) {
        if (!h->side && (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
                         cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                         cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess))
            return LEDDS_ECUDA;
        if (cudaEventRecord(h->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(h->side, h->ev_fork, 0) != cudaSuccess)
            return LEDDS_ECUDA;
        st = h->side;
    }
    ledds_prof_start(LEDDS_K_DEM_SORT, st);
    int hb = (n + SORT_THREADS * 8 - 1) / (SORT_THREADS * 8);
    if (hb > ledds_sm_count() * 8) hb = ledds_sm_count() * 8;
    uint32_t* unsorted = at<uint32_t>(scratch, s.tile_counter) + 7;          // zeroed with the tickets
    const int always = (h->p.sort_every_step || h->counting) ? 1 : 0;
    if (h->counting) {
        // counting sort: the drift kernel has counted; cell counts -> cell ranges, then every particle to start + its number
        launch_pdl(dem_cell_scan_kernel, dim3(h->cell_tiles), dim3(SCAN_THREADS), 0, st, n, (uint32_t)d.ncell, cells,
                   at<uint32_t>(scratch, s.cell_scan_state), at<uint32_t>(scratch, s.tile_counter) + 5);
        LEDDS_CHECK_LAUNCH();
        launch_pdl(dem_scatter_kernel, dim3(nb), dim3(tb), 0, st, n, at<uint32_t>(scratch, s.key[0]), at<uint32_t>(scratch, s.idx[0]),
                   cells, at<uint32_t>(scratch, s.hid), at<uint32_t>(scratch, s.key[1]), at<uint32_t>(scratch, s.idx[1]),
                   at<uint32_t>(scratch, s.sid_tmp));
        LEDDS_CHECK_LAUNCH();
    } else {
    launch_pdl(dem_hist_kernel, dim3(hb), dim3(SORT_THREADS), 0, st, at<uint32_t>(scratch, s.key[0]), n, h->passes,
                                                 at<uint32_t>(scratch, s.hist_digit), unsorted);
    LEDDS_CHECK_LAUNCH();
    for (int p = 0; p < h->passes; ++p) {
        const int in = p & 1, out = in ^ 1;
        launch_pdl(dem_onesweep_kernel, dim3(h->tiles), dim3(SORT_THREADS), 0, st, 
            at<uint32_t>(scratch, s.key[in]), at<uint32_t>(scratch, s.idx[in]), at<uint32_t>(scratch, s.key[out]),
            at<uint32_t>(scratch, s.idx[out]), n, 8 * p, at<uint32_t>(scratch, s.hist_digit) + p * SORT_RADIX,
            at<uint32_t>(scratch, s.tile_state) + (size_t)p * h->tiles * SORT_RADIX,
            at<uint32_t>(scratch, s.tile_counter) + p, unsorted, always);
        LEDDS_CHECK_LAUNCH();
    }
    }
    ledds_prof_stop(LEDDS_K_DEM_SORT, st);
    h->sorted_buf = h->counting ? 1 : (h->passes & 1);
    h->sh_buf = 1 - h->sorted_buf;                             // the other idx buffer is free once the last pass / the scatter is done
    h->have_sort = true;
    const uint32_t* key_home = at<uint32_t>(scratch, s.key[0]);
    const uint32_t* key_sorted = at<uint32_t>(scratch, s.key[h->sorted_buf]);
    const uint32_t* idx_sorted = at<uint32_t>(scratch, s.idx[h->sorted_buf]);
    uint32_t* skey = at<uint32_t>(scratch, s.skey_f);
    uint32_t* sh = at<uint32_t>(scratch, s.idx[h->sh_buf]);
    uint32_t* sid = at<uint32_t>(scratch, s.sid);
    uint32_t* nfwd = at<uint32_t>(scratch, s.nfwd);
    uint32_t* nback = at<uint32_t>(scratch, s.nback);
    uint32_t* off = at<uint32_t>(scratch, s.off);
    ledds_prof_start(LEDDS_K_DEM_GATHER, st);
    if (!h->counting) {                                        // (the counting sort has made the cell ranges and sid_tmp itself)
        launch_pdl(dem_ranges_kernel, dim3(nb), dim3(tb), 0, st, n, key_home, key_sorted, idx_sorted, unsorted, always,
                   at<uint32_t>(scratch, s.hid), at<uint32_t>(scratch, s.sid_tmp), at<uint2>(scratch, s.cell_range));
        LEDDS_CHECK_LAUNCH();
    }
    launch_pdl(dem_gather_kernel<T>, dim3(nb), dim3(tb), 0, st, d, key_home, key_sorted, idx_sorted, unsorted, always, skey,
               at<uint32_t>(scratch, s.sid_tmp), at<uint2>(scratch, s.cell_range), at<typename Real<T>::v4>(scratch, s.hx),
               at<typename Real<T>::v4>(scratch, s.xr_s), at<float4>(scratch, s.xf_s), sid, sh, nback);
    ledds_prof_stop(LEDDS_K_DEM_GATHER, st);
    LEDDS_CHECK_LAUNCH();
    const int prev = h->cur, nw = 1 - h->cur;
    ledds_prof_start(LEDDS_K_DEM_CONTACT, st);
    const int cb = (n + CONTACT_BLOCK - 1) / CONTACT_BLOCK;
    if (d.bc[0] && d.bc[1] && d.bc[2])
        launch_pdl(dem_detect_kernel<T, false>, dim3(cb), dim3(CONTACT_BLOCK), 0, st, d, skey, at<typename Real<T>::v4>(scratch, s.xr_s), at<float4>(scratch, s.xf_s),
                                                                        at<uint2>(scratch, s.cell_range), nfwd, nback, at<uint32_t>(scratch, s.cand), status);
    else
        launch_pdl(dem_detect_kernel<T, true>, dim3(cb), dim3(CONTACT_BLOCK), 0, st, d, skey, at<typename Real<T>::v4>(scratch, s.xr_s), at<float4>(scratch, s.xf_s),
                                                                       at<uint2>(scratch, s.cell_range), nfwd, nback, at<uint32_t>(scratch, s.cand), status);
    LEDDS_CHECK_LAUNCH();
    launch_pdl(dem_scan_kernel, dim3(h->scan_tiles), dim3(SCAN_THREADS), 0, st, n, (uint32_t)d.maxc, nfwd, nback, off, at<uint32_t>(scratch, s.scan_state),
                                                            at<uint32_t>(scratch, s.tile_counter) + 4);
    LEDDS_CHECK_LAUNCH();
    const DemEnds E = {at<uint32_t>(scratch, s.end_s), at<uint32_t>(scratch, s.end_t), at<uint32_t>(scratch, s.end_hs),
                       at<uint32_t>(scratch, s.end_ht), at<uint32_t>(scratch, s.end_prev)};
    launch_pdl(dem_fill_kernel<T>, dim3(cb), dim3(CONTACT_BLOCK), (size_t)d.maxc * CONTACT_BLOCK * 12, st, 
        n, (uint32_t)d.maxc, nfwd, nback, at<uint32_t>(scratch, s.cand), sid, sh, off, row, fm, at<uint32_t>(history, hs.hq[prev]), E,
        at<uint32_t>(history, hs.hq[nw]), status);
    LEDDS_CHECK_LAUNCH();
    void (*force_kernel)(const DemDevT<T>, const typename Real<T>::v4*, const T*, const uint32_t*, const DemEnds, const uint32_t*, T*, const T*, T*,
                         int32_t*, T) = h->p.model == 1 ? dem_force_kernel<T, true> : dem_force_kernel<T, false>;
    launch_pdl(force_kernel, dim3((n + FORCE_PB - 1) / FORCE_PB), dim3(FORCE_THREADS), 0, st, 
        d, at<typename Real<T>::v4>(scratch, s.xr_s), at<T>(scratch, s.pvw), off, E, sh, fm, at<T>(history, hs.hdt[prev]),
        at<T>(history, hs.hdt[nw]), status, (T)dt_hist);
    ledds_prof_stop(LEDDS_K_DEM_CONTACT, st);
    LEDDS_CHECK_LAUNCH();
    h->cur = nw;
    if (fork && cudaEventRecord(h->ev_join, st) != cudaSuccess) return LEDDS_ECUDA;
    return LEDDS_OK;
}

template <typename T>
static int dem_kick_t(ledds_dem* h, const T* f_ext, const T* m_ext, const void* history, void* scratch, cudaStream_t st)
{
    const int n = h->d.n;
    if (n == 0) return LEDDS_OK;
    const DemScratch& s = h->s;
    ledds_prof_start(LEDDS_K_DEM_KICK, st);
    dem_kick_kernel<T><<<(unsigned)((3ll * n + 255) / 256), 256, 0, st>>>(dem_dev<T>(h), at<typename Real<T>::v4>(scratch, s.hx), at<uint32_t>(scratch, s.hid),
                                                                       at<T>(history, h->hs.fm[h->rec]), f_ext, m_ext,
                                                                       at<T>(scratch, s.hv), at<T>(scratch, s.hw),
                                                                       at<T>(scratch, s.ha), at<T>(scratch, s.hal), 0);
    ledds_prof_stop(LEDDS_K_DEM_KICK, st);
    LEDDS_CHECK_LAUNCH();
    return LEDDS_OK;
}

template <typename T>
static int dem_init_t(ledds_dem** out, const ledds_dem_params* p, const T* x, const T* v,
                              const T* w, const T* radius, T* a, T* alpha, void* history,
                              void* scratch, int32_t* status, void* stream)
{
    if (!out || !p || !status) return LEDDS_EINVAL;
    if (p->n != 0 && (!x || !v || !w || !radius || !a || !alpha || !history || !scratch)) return LEDDS_EINVAL;
    const void* ptrs[] = {x, v, w, radius, a, alpha, history, scratch, status};
    for (const void* q : ptrs)
        if (!ledds_aligned16(q)) return LEDDS_EALIGN;
    ledds_dem* h = new (std::nothrow) ledds_dem();
    if (!h) return LEDDS_EINVAL;
    int rc = dem_setup(p, h, sizeof(T));
    if (rc) { delete h; return rc; }
    cudaStream_t st = (cudaStream_t)stream;
    if ((h->hs.total && cudaMemsetAsync(history, 0, h->hs.total, st) != cudaSuccess) ||
        cudaMemsetAsync(status, 0, 16, st) != cudaSuccess) {
        delete h;
        return LEDDS_ECUDA;
    }
    // forces of the initial state: no drift, delta_t stays 0 (dt_hist = 0); a(0), alpha(0) back to the caller
    rc = dem_import_t<T>(h, x, v, w, (const T*)nullptr, (const T*)nullptr, radius, history, scratch, st);
    if (!rc) rc = dem_advance_t<T>(h, history, scratch, status, 0.0, false, st, false, nullptr);
    if (rc) { delete h; return rc; }
    if (h->d.n == 0) { *out = h; return LEDDS_OK; }
    const DemScratch& s = h->s;
    dem_kick_kernel<T><<<(unsigned)((3ll * h->d.n + 255) / 256), 256, 0, st>>>(dem_dev<T>(h), at<typename Real<T>::v4>(scratch, s.hx), at<uint32_t>(scratch, s.hid),
                                                                            at<T>(history, h->hs.fm[h->rec]), (const T*)nullptr, (const T*)nullptr,
                                                                            at<T>(scratch, s.hv), at<T>(scratch, s.hw),
                                                                            at<T>(scratch, s.ha), at<T>(scratch, s.hal), 1);
    ledds_count_launch(1);
    if (cudaPeekAtLastError() != cudaSuccess) { delete h; return LEDDS_ECUDA; }
    rc = dem_export_t<T>(h, (T*)nullptr, (T*)nullptr, (T*)nullptr, a, alpha, scratch, st);
    if (rc) { delete h; return rc; }
    *out = h;
    return LEDDS_OK;
}

// steps between two re-homings inside one long call (the home order goes stale as particles change cells)
#define DEM_REHOME_STEPS 256

template <typename T>
static int dem_step_t(ledds_dem* h, T* x, T* v, T* w, T* a, T* alpha,
                              const T* radius, const T* f_ext, const T* m_ext, void* history,
                              void* scratch, int32_t* status, int nsteps, void* stream)
{
    if (!h || !status || nsteps < 0 || h->f32 != (sizeof(T) == 4)) return LEDDS_EINVAL;   // the handle fixes the real type
    if (h->d.n == 0 || nsteps == 0) return LEDDS_OK;
    if (!x || !v || !w || !a || !alpha || !radius || !history || !scratch) return LEDDS_EINVAL;
    const void* ptrs[] = {x, v, w, a, alpha, radius, f_ext, m_ext, history, scratch, status};
    for (const void* q : ptrs)
        if (!ledds_aligned16(q)) return LEDDS_EALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    const DemKickT<T> kick = {f_ext, m_ext};
    int rc = dem_import_t<T>(h, x, v, w, a, alpha, radius, history, scratch, st);
    if (rc) return rc;
    for (int s = 0; s < nsteps; ++s) {
        // the kick of step s - 1 rides on the drift of step s; only the last step of the call (and the one before
        // a re-homing) kicks on its own
        const bool rehome = s > 0 && s % DEM_REHOME_STEPS == 0;
        if (rehome) {
            rc = dem_kick_t<T>(h, f_ext, m_ext, history, scratch, st);
            if (!rc) rc = dem_export_t<T>(h, x, v, w, a, alpha, scratch, st);
            if (!rc) rc = dem_import_t<T>(h, x, v, w, a, alpha, radius, history, scratch, st);
            if (rc) return rc;
        }
        const DemKickT<T>* first = (s > 0 && !rehome) ? &kick : nullptr;
        int batch = 1;                                         // small systems: all steps up to the next re-homing in one launch
        if (dem_small_ok(h)) batch = std::min(nsteps - s, DEM_REHOME_STEPS - s % DEM_REHOME_STEPS);
        if (batch > 1) rc = dem_small_advance<T>(h, history, scratch, status, h->d.dt, true, st, false, first, batch, &kick);
        else rc = dem_advance_t<T>(h, history, scratch, status, h->d.dt, true, st, false, first);
        if (rc) return rc;
        h->steps += batch;
        s += batch - 1;
    }
    rc = dem_kick_t<T>(h, f_ext, m_ext, history, scratch, st);
    if (rc) return rc;
    return dem_export_t<T>(h, x, v, w, a, alpha, scratch, st);
}

template <typename T>
static int dem_query_t(ledds_dem* h, const void* history, const void* scratch, uint32_t* sorted_idx,
                               uint32_t* sorted_key, uint32_t* pairs, T* pair_dt, uint32_t pair_cap,
                               uint32_t* n_pairs, T* force, T* torque, void* stream)
{
    if (!h || h->f32 != (sizeof(T) == 4)) return LEDDS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)h->d.n;
    if (n == 0) {
        if (n_pairs && cudaMemsetAsync(n_pairs, 0, sizeof(uint32_t), st) != cudaSuccess) return LEDDS_ECUDA;
        return LEDDS_OK;
    }
    if (!history || !scratch) return LEDDS_EINVAL;
    const DemScratch& s = h->s;
    const DemHistory& hs = h->hs;
    auto copy = [&](void* dst, const void* src, size_t bytes) {
        return !dst || cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, st) == cudaSuccess;
    };
    if (!copy(sorted_idx, at<char>(scratch, s.sid), n * 4) ||
        !copy(sorted_key, at<char>(scratch, s.skey_f), n * 4))
        return LEDDS_ECUDA;
    const int tb = 128, nb = ((int)n + tb - 1) / tb;
    if (force || torque) {
        dem_unpack_fm_kernel<T><<<nb, tb, 0, st>>>((int)n, at<uint32_t>(scratch, s.hid), at<T>(history, hs.fm[h->rec]), force, torque);
        LEDDS_CHECK_LAUNCH();
    }
    if (pairs || pair_dt || n_pairs) {
        // scratch is logically const for the caller; the query arrays are ours to overwrite
        uint32_t* cnt = const_cast<uint32_t*>(at<uint32_t>(scratch, s.pair_count));
        uint32_t* poff = const_cast<uint32_t*>(at<uint32_t>(scratch, s.pair_off));
        uint32_t* pos = const_cast<uint32_t*>(at<uint32_t>(scratch, s.pos_of_id));
        const uint32_t* off = at<uint32_t>(scratch, s.off);
        const uint32_t* hq = at<uint32_t>(history, hs.hq[h->cur]);
        dem_query_pos_kernel<<<nb, tb, 0, st>>>((int)n, at<uint32_t>(scratch, s.sid), pos);
        dem_pair_count_kernel<<<nb, tb, 0, st>>>((int)n, pos, off, hq, cnt);
        dem_block_scan_kernel<<<1, 1024, 0, st>>>((int)n, cnt, poff);
        dem_pair_write_kernel<T><<<nb, tb, 0, st>>>((int)n, pos, off, hq, at<T>(history, hs.hdt[h->cur]), poff, pair_cap, pairs,
                                                 pair_dt, n_pairs);
        ledds_count_launch(3);
        LEDDS_CHECK_LAUNCH();
    }
    return LEDDS_OK;
}

// ---- entry points: the fp64 set, the fp32 set (include/ledds.h), and the fp64 pieces coupled.cu drives
extern "C" int ledds_dem_init(ledds_dem** out, const ledds_dem_params* p, const double* x, const double* v, const double* w,
                              const double* radius, double* a, double* alpha, void* history, void* scratch, int32_t* status,
                              void* stream)
{
    return dem_init_t<double>(out, p, x, v, w, radius, a, alpha, history, scratch, status, stream);
}
extern "C" int ledds_dem_init_f32(ledds_dem** out, const ledds_dem_params* p, const float* x, const float* v, const float* w,
                                  const float* radius, float* a, float* alpha, void* history, void* scratch, int32_t* status,
                                  void* stream)
{
    return dem_init_t<float>(out, p, x, v, w, radius, a, alpha, history, scratch, status, stream);
}
extern "C" int ledds_dem_step(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha, const double* radius,
                              const double* f_ext, const double* m_ext, void* history, void* scratch, int32_t* status,
                              int nsteps, void* stream)
{
    return dem_step_t<double>(h, x, v, w, a, alpha, radius, f_ext, m_ext, history, scratch, status, nsteps, stream);
}
extern "C" int ledds_dem_step_f32(ledds_dem* h, float* x, float* v, float* w, float* a, float* alpha, const float* radius,
                                  const float* f_ext, const float* m_ext, void* history, void* scratch, int32_t* status,
                                  int nsteps, void* stream)
{
    return dem_step_t<float>(h, x, v, w, a, alpha, radius, f_ext, m_ext, history, scratch, status, nsteps, stream);
}
extern "C" int ledds_dem_query(ledds_dem* h, const void* history, const void* scratch, uint32_t* sorted_idx,
                               uint32_t* sorted_key, uint32_t* pairs, double* pair_dt, uint32_t pair_cap, uint32_t* n_pairs,
                               double* force, double* torque, void* stream)
{
    return dem_query_t<double>(h, history, scratch, sorted_idx, sorted_key, pairs, pair_dt, pair_cap, n_pairs, force, torque, stream);
}
extern "C" int ledds_dem_query_f32(ledds_dem* h, const void* history, const void* scratch, uint32_t* sorted_idx,
                                   uint32_t* sorted_key, uint32_t* pairs, float* pair_dt, uint32_t pair_cap, uint32_t* n_pairs,
                                   float* force, float* torque, void* stream)
{
    return dem_query_t<float>(h, history, scratch, sorted_idx, sorted_key, pairs, pair_dt, pair_cap, n_pairs, force, torque, stream);
}

int ledds_dem_import(ledds_dem* h, const double* x, const double* v, const double* w, const double* a, const double* alpha,
                     const double* radius, void* history, void* scratch, cudaStream_t st)
{
    return h->f32 ? LEDDS_EINVAL : dem_import_t<double>(h, x, v, w, a, alpha, radius, history, scratch, st);
}
int ledds_dem_export(ledds_dem* h, double* x, double* v, double* w, double* a, double* alpha, const void* scratch, cudaStream_t st)
{
    return dem_export_t<double>(h, x, v, w, a, alpha, scratch, st);
}
int ledds_dem_advance_contacts(ledds_dem* h, void* history, void* scratch, int32_t* status, double dt_hist, bool drift,
                               cudaStream_t st, bool fork, const DemKick* kick)
{
    return dem_advance_t<double>(h, history, scratch, status, dt_hist, drift, st, fork, kick);
}
int ledds_dem_kick(ledds_dem* h, const double* f_ext, const double* m_ext, const void* history, void* scratch, cudaStream_t st)
{
    return dem_kick_t<double>(h, f_ext, m_ext, history, scratch, st);
}

extern "C" int ledds_dem_destroy(ledds_dem* h)
{
    if (h && h->side) {
        cudaStreamDestroy(h->side);
        cudaEventDestroy(h->ev_fork);
        cudaEventDestroy(h->ev_join);
    }
    delete h;
    return LEDDS_OK;
}

// ------------------------------------------------------------------------------ cell order without any allocation
// ledds_dem_cell_order_static (include/ledds.h): the key + radix-sort stage of the pipeline above for callers that can
// neither allocate nor bring a scratch buffer (graph capture, serving loops).  Its scratch -- digit histograms, tile
// tickets, look-back descriptors and the ping-pong key / index buffers -- is this file-scope device array; every GPU
// that loads the library holds its STATIC_SCRATCH_BYTES (about 4.4 MiB) until the process exits.  All calls on a device
// share it: calls that overlap on the GPU race (see the header).
#include <mutex>

#define STATIC_MAX_N LEDDS_CELL_ORDER_STATIC_MAX_N
#define STATIC_MAX_TILES ((STATIC_MAX_N + SORT_TILE - 1) / SORT_TILE)
#define STATIC_OFF_HIST 0                                                         /* uint32 [4][256]             */
#define STATIC_OFF_TICKET (STATIC_OFF_HIST + 4 * SORT_RADIX * 4)                  /* uint32 [8] (+ padding)      */
#define STATIC_OFF_STATE (STATIC_OFF_TICKET + 256)                                /* uint32 [4][max tiles][256]  */
#define STATIC_OFF_KEY (STATIC_OFF_STATE + 4 * STATIC_MAX_TILES * SORT_RADIX * 4) /* uint32 [2][max n]           */
#define STATIC_OFF_IDX (STATIC_OFF_KEY + 2 * STATIC_MAX_N * 4)                    /* uint32 [2][max n]           */
#define STATIC_SCRATCH_BYTES (STATIC_OFF_IDX + 2 * STATIC_MAX_N * 4)
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

// In host code g_static_scratch is only a stand-in for the symbol: its device address is asked for once per device,
// with that device current, and kept here.
#define STATIC_MAX_DEVICES 64
static unsigned char* g_static_ptr[STATIC_MAX_DEVICES];
static std::mutex g_static_mutex;

static int dem_static_scratch(unsigned char** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return LEDDS_ECUDA;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return LEDDS_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) return LEDDS_ECUDA;
        g_static_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_ptr[dev];
    return LEDDS_OK;
}

// cell key of every particle from the caller's positions (same expressions as dem_drift_key_kernel), value = id
__global__ void __launch_bounds__(DRIFT_BLOCK) dem_key_of_x_kernel(const DemDev P, const double* __restrict__ x,
                                                                   uint32_t* __restrict__ key, uint32_t* __restrict__ idx)
{
    const int i = blockIdx.x * DRIFT_BLOCK + threadIdx.x;
    if (i >= P.n) return;
    const int cx = dem_cell_coord(P, x[3 * (size_t)i], 0), cy = dem_cell_coord(P, x[3 * (size_t)i + 1], 1),
              cz = dem_cell_coord(P, x[3 * (size_t)i + 2], 2);
    key[i] = (uint32_t)(cx + P.nc[0] * (cy + P.nc[1] * cz));
    idx[i] = (uint32_t)i;
}

extern "C" int ledds_dem_cell_order_static_max_n(void) { return STATIC_MAX_N; }

extern "C" int ledds_dem_cell_order_static(const ledds_dem_params* p, const double* x, uint32_t* sorted_idx,
                                           uint32_t* sorted_key, void* stream)
{
    if (!p) return LEDDS_EINVAL;
    if (p->n > STATIC_MAX_N) return LEDDS_ECAPACITY;           // the static scratch holds STATIC_MAX_N particles, no more
    ledds_dem tmp;
    const int rc = dem_setup(p, &tmp, 8);
    if (rc) return rc;
    const int n = p->n;
    if (n == 0) return LEDDS_OK;
    if (!x || !sorted_idx || !sorted_key) return LEDDS_EINVAL;
    if (((uintptr_t)x | (uintptr_t)sorted_idx | (uintptr_t)sorted_key) & 15) return LEDDS_EALIGN;
    unsigned char* base = nullptr;
    const int rs = dem_static_scratch(&base);
    if (rs) return rs;
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t* hist = reinterpret_cast<uint32_t*>(base + STATIC_OFF_HIST);
    uint32_t* ticket = reinterpret_cast<uint32_t*>(base + STATIC_OFF_TICKET);
    uint32_t* state = reinterpret_cast<uint32_t*>(base + STATIC_OFF_STATE);
    uint32_t* key[2] = {reinterpret_cast<uint32_t*>(base + STATIC_OFF_KEY), reinterpret_cast<uint32_t*>(base + STATIC_OFF_KEY) + STATIC_MAX_N};
    uint32_t* idx[2] = {reinterpret_cast<uint32_t*>(base + STATIC_OFF_IDX), reinterpret_cast<uint32_t*>(base + STATIC_OFF_IDX) + STATIC_MAX_N};
    // the array keeps what the last call left: histograms, tickets and descriptors must start at zero
    if (cudaMemsetAsync(base + STATIC_OFF_HIST, 0, STATIC_OFF_STATE + (size_t)4 * tmp.tiles * SORT_RADIX * 4, st) != cudaSuccess)
        return LEDDS_ECUDA;
    dem_key_of_x_kernel<<<(n + DRIFT_BLOCK - 1) / DRIFT_BLOCK, DRIFT_BLOCK, 0, st>>>(tmp.d, x, key[0], idx[0]);
    LEDDS_CHECK_LAUNCH();
    int hb = (n + SORT_THREADS * 8 - 1) / (SORT_THREADS * 8);
    if (hb > ledds_sm_count() * 8) hb = ledds_sm_count() * 8;
    uint32_t* unsorted = ticket + 7;
    dem_hist_kernel<<<hb, SORT_THREADS, 0, st>>>(key[0], n, tmp.passes, hist, unsorted);
    LEDDS_CHECK_LAUNCH();
    // the input is in id order and every pass is stable: the result is ordered by (cell key, id) as it stands.  The
    // last pass writes into the caller's arrays.
    for (int q = 0; q < tmp.passes; ++q) {
        const int in = q & 1, out = in ^ 1;
        const bool last = q == tmp.passes - 1;
        dem_onesweep_kernel<<<tmp.tiles, SORT_THREADS, 0, st>>>(key[in], idx[in], last ? sorted_key : key[out],
                                                                last ? sorted_idx : idx[out], n, 8 * q, hist + q * SORT_RADIX,
                                                                state + (size_t)q * tmp.tiles * SORT_RADIX, ticket + q, unsorted, 1);
        LEDDS_CHECK_LAUNCH();
    }
    return LEDDS_OK;
}
