// D3Q19 BGK fused stream-collide for sm_100a (Eq. 22-28; boundaries PAPER.md:254).
//
// State = pre-collision populations in canonical layout f[q][z][y][x] (x fastest), two lattices.
// One pass reads 19 doubles and writes 19 doubles per cell: 304 B/cell of algorithmic traffic.
// One kernel: one cell per thread, aligned coalesced loads, stores shifted by c_q ("push"); measured on B200 it
// runs at the HBM copy rate, so no second variant is kept (a row-rotating kernel with aligned stores was measured
// in round 1 and was not faster).
#include <new>

#include "lbm_kernels.cuh"

// ------------------------------------------------------------------------------------ helpers
template <typename T>
__global__ void lbm_init_eq_kernel(T* __restrict__ f, const T* __restrict__ rho, const T* __restrict__ u, long long N)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= N) return;
    const T r = rho ? rho[c] : T(1);
    const T ux = u ? u[c] : T(0), uy = u ? u[N + c] : T(0), uz = u ? u[2 * N + c] : T(0);
    T fe[LEDDS_Q];
    lb_equilibrium(fe, r, ux, uy, uz);
#pragma unroll
    for (int q = 0; q < LEDDS_Q; ++q) f[(long long)q * N + c] = fe[q];
}

template <typename T>
__global__ void lbm_export_kernel(const T* __restrict__ f, T* __restrict__ fc, T* __restrict__ rho, T* __restrict__ u,
                                  long long N)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= N) return;
    T v[LEDDS_Q];
#pragma unroll
    for (int q = 0; q < LEDDS_Q; ++q) v[q] = f[(long long)q * N + c];
    if (fc) {
#pragma unroll
        for (int q = 0; q < LEDDS_Q; ++q) fc[(long long)q * N + c] = v[q];
    }
    if (rho || u) {
        T r, ux, uy, uz;
        lb_moments(v, r, ux, uy, uz);
        if (rho) rho[c] = r;
        if (u) { u[c] = ux; u[N + c] = uy; u[2 * N + c] = uz; }
    }
}

// ------------------------------------------------------------------------------------ stream-collide
// Block = 128 threads = BX cells along x times 128 / BX rows along y (BX = 128 unless the lattice is narrower,
// so that narrow lattices do not run half-empty blocks); a warp always lies inside one row.
template <typename T, typename I, int BX, bool TRT>
__global__ void __launch_bounds__(128) lbm_push_kernel(const T* __restrict__ fin, T* __restrict__ fout,
                                                       const __grid_constant__ LbmDev P)
{
    const int x = blockIdx.x * BX + (int)(threadIdx.x % BX);
    const int y = blockIdx.y * (128 / BX) + (int)(threadIdx.x / BX), z = blockIdx.z;
    if (x >= P.nx || y >= P.ny) return;
    const I cell = ((I)z * (I)P.ny + (I)y) * (I)P.nx + (I)x;
    T f[LEDDS_Q];
    lb_load<I>(fin, (I)P.N, cell, f);
    T rho, ux, uy, uz;
    lb_moments(f, rho, ux, uy, uz);
    lb_collide<TRT>(f, P, rho, ux, uy, uz);
    lb_push_store<I>(fout, P, x, y, z, f, rho);
}

template <typename T, typename I, bool TRT>
static void lbm_push_launch(const T* src, T* dst, const LbmDev& d, cudaStream_t st)
{
    const int bx = lb_block_x(d.nx), rows = 128 / bx;
    const dim3 block(128), grid((d.nx + bx - 1) / bx, (d.ny + rows - 1) / rows, d.nz);
    if (bx == 128) lbm_push_kernel<T, I, 128, TRT><<<grid, block, 0, st>>>(src, dst, d);
    else if (bx == 64) lbm_push_kernel<T, I, 64, TRT><<<grid, block, 0, st>>>(src, dst, d);
    else lbm_push_kernel<T, I, 32, TRT><<<grid, block, 0, st>>>(src, dst, d);
}

// ------------------------------------------------------------------------------------ host API
static int lbm_validate(const ledds_lbm_params* p)
{
    if (!p) return LEDDS_EINVAL;
    if (p->nx < 1 || p->ny < 1 || p->nz < 1) return LEDDS_EINVAL;
    if ((long long)p->nx * p->ny * p->nz > (1ll << 31)) return LEDDS_EINVAL;
    if (!(p->tau > 0.5)) return LEDDS_EINVAL;
    if (p->layout != 0) return LEDDS_EINVAL;
    if (p->variant != 0 && p->variant != 1 && p->variant != 3) return LEDDS_EINVAL;
    if (p->collision != 0 && p->collision != 1) return LEDDS_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (p->bc[a] != 0 && p->bc[a] != 1) return LEDDS_EINVAL;
    // a periodic axis of length 1 would stream a population onto itself: allowed (it is a no-op wrap)
    return LEDDS_OK;
}

// ---- the calls are written once for both precisions; T = float is the _f32 set of entry points
template <typename T>
static int lbm_workspace_bytes_t(const ledds_lbm_params* p, size_t* f_bytes)
{
    const int rc = lbm_validate(p);
    if (rc) return rc;
    if (!f_bytes) return LEDDS_EINVAL;
    *f_bytes = (size_t)2 * LEDDS_Q * p->nx * p->ny * p->nz * sizeof(T);
    return LEDDS_OK;
}

template <typename T>
static int lbm_init_t(ledds_lbm** out, const ledds_lbm_params* p, T* f, const T* rho, const T* u, void* stream)
{
    const int rc = lbm_validate(p);
    if (rc) return rc;
    if (!out || !f) return LEDDS_EINVAL;
    if (!ledds_aligned16(f) || !ledds_aligned16(rho) || !ledds_aligned16(u)) return LEDDS_EALIGN;
    ledds_lbm* h = new (std::nothrow) ledds_lbm();
    if (!h) return LEDDS_EINVAL;
    h->p = *p;
    h->f32 = sizeof(T) == 4;
    LbmDev& d = h->d;
    d.nx = p->nx; d.ny = p->ny; d.nz = p->nz;
    d.N = (long long)p->nx * p->ny * p->nz;
    d.tau = p->tau;
    d.omega = 1.0 / p->tau;
    d.omega_minus = 8.0 * (2.0 - d.omega) / (8.0 - d.omega);                  // Eq. (31)
    d.trt = p->collision;
    d.any_wall_velocity = 0;
    for (int a = 0; a < 3; ++a) {
        d.bc[a] = p->bc[a];
        for (int s = 0; s < 2; ++s)
            for (int c = 0; c < 3; ++c) {
                d.uw[(a * 2 + s) * 3 + c] = p->u_wall[a][s][c];
                if (p->bc[a] && p->u_wall[a][s][c] != 0.0) d.any_wall_velocity = 1;
            }
    }
    h->parity = 0;
    h->steps = 0;
    const int tb = 256;
    lbm_init_eq_kernel<T><<<(unsigned)((d.N + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(f, rho, u, d.N);
    ledds_count_launch(1);
    if (cudaPeekAtLastError() != cudaSuccess) { delete h; return LEDDS_ECUDA; }
    *out = h;
    return LEDDS_OK;
}

template <typename T>
static bool lbm_handle_is(const ledds_lbm* h) { return h && h->f32 == (sizeof(T) == 4); }

template <typename T>
static int lbm_import_t(ledds_lbm* h, T* f, const T* fc, void* stream)
{
    if (!lbm_handle_is<T>(h) || !f || !fc) return LEDDS_EINVAL;
    if (!ledds_aligned16(f) || !ledds_aligned16(fc)) return LEDDS_EALIGN;
    T* cur = f + (size_t)h->parity * LEDDS_Q * h->d.N;
    if (cudaMemcpyAsync(cur, fc, sizeof(T) * LEDDS_Q * h->d.N, cudaMemcpyDeviceToDevice, (cudaStream_t)stream) != cudaSuccess)
        return LEDDS_ECUDA;
    return LEDDS_OK;
}

// one stream-collide launch src -> dst (used by ledds_lbm_step; coupled.cu has its own PSM launch)
template <typename T>
static int lbm_launch(const ledds_lbm* h, const T* src, T* dst, cudaStream_t st)
{
    const LbmDev& d = h->d;
    if (d.ny > 65535 || d.nz > 65535) return LEDDS_EINVAL;
    const bool u32 = lb_fits_u32(d.N) && h->p.variant != 3;   // 3 = 64-bit indices whatever the size
    ledds_prof_start(LEDDS_K_LBM, st);
    if (u32 && !d.trt) lbm_push_launch<T, unsigned, false>(src, dst, d, st);
    else if (u32) lbm_push_launch<T, unsigned, true>(src, dst, d, st);
    else if (!d.trt) lbm_push_launch<T, long long, false>(src, dst, d, st);
    else lbm_push_launch<T, long long, true>(src, dst, d, st);
    ledds_prof_stop(LEDDS_K_LBM, st);
    LEDDS_CHECK_LAUNCH();
    return LEDDS_OK;
}

template <typename T>
static int lbm_step_t(ledds_lbm* h, T* f, int nsteps, void* stream)
{
    if (!lbm_handle_is<T>(h) || !f || nsteps < 0) return LEDDS_EINVAL;
    if (!ledds_aligned16(f)) return LEDDS_EALIGN;
    const size_t half = (size_t)LEDDS_Q * h->d.N;
    for (int s = 0; s < nsteps; ++s) {
        const int rc = lbm_launch<T>(h, f + h->parity * half, f + (1 - h->parity) * half, (cudaStream_t)stream);
        if (rc) return rc;
        h->parity ^= 1;
        h->steps++;
    }
    return LEDDS_OK;
}

template <typename T>
static int lbm_export_t(ledds_lbm* h, const T* f, T* fc, T* rho, T* u, void* stream)
{
    if (!lbm_handle_is<T>(h) || !f) return LEDDS_EINVAL;
    if (!ledds_aligned16(f) || !ledds_aligned16(fc) || !ledds_aligned16(rho) || !ledds_aligned16(u)) return LEDDS_EALIGN;
    const int tb = 256;
    lbm_export_kernel<T><<<(unsigned)((h->d.N + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(
        f + (size_t)h->parity * LEDDS_Q * h->d.N, fc, rho, u, h->d.N);
    LEDDS_CHECK_LAUNCH();
    return LEDDS_OK;
}

extern "C" int ledds_lbm_workspace_bytes(const ledds_lbm_params* p, size_t* f_bytes) { return lbm_workspace_bytes_t<double>(p, f_bytes); }
extern "C" int ledds_lbm_workspace_bytes_f32(const ledds_lbm_params* p, size_t* f_bytes) { return lbm_workspace_bytes_t<float>(p, f_bytes); }

extern "C" int ledds_lbm_init(ledds_lbm** out, const ledds_lbm_params* p, double* f, const double* rho, const double* u,
                              void* stream)
{
    return lbm_init_t<double>(out, p, f, rho, u, stream);
}
extern "C" int ledds_lbm_init_f32(ledds_lbm** out, const ledds_lbm_params* p, float* f, const float* rho, const float* u,
                                  void* stream)
{
    return lbm_init_t<float>(out, p, f, rho, u, stream);
}

extern "C" const double* ledds_lbm_current(const ledds_lbm* h, const double* f)
{
    return (lbm_handle_is<double>(h) && f) ? f + (size_t)h->parity * LEDDS_Q * h->d.N : nullptr;
}

extern "C" int ledds_lbm_import(ledds_lbm* h, double* f, const double* fc, void* stream) { return lbm_import_t<double>(h, f, fc, stream); }
extern "C" int ledds_lbm_import_f32(ledds_lbm* h, float* f, const float* fc, void* stream) { return lbm_import_t<float>(h, f, fc, stream); }

extern "C" int ledds_lbm_step(ledds_lbm* h, double* f, int nsteps, void* stream) { return lbm_step_t<double>(h, f, nsteps, stream); }
extern "C" int ledds_lbm_step_f32(ledds_lbm* h, float* f, int nsteps, void* stream) { return lbm_step_t<float>(h, f, nsteps, stream); }

extern "C" int ledds_lbm_export(ledds_lbm* h, const double* f, double* fc, double* rho, double* u, void* stream)
{
    return lbm_export_t<double>(h, f, fc, rho, u, stream);
}
extern "C" int ledds_lbm_export_f32(ledds_lbm* h, const float* f, float* fc, float* rho, float* u, void* stream)
{
    return lbm_export_t<float>(h, f, fc, rho, u, stream);
}

extern "C" int ledds_lbm_destroy(ledds_lbm* h)
{
    delete h;
    return LEDDS_OK;
}

extern "C" const char* ledds_version(void) { return "ledds-b200 0.2 (sm_100a, fp64; fp32 lattice optional)"; }
