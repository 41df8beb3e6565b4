// Device-side building blocks of the D3Q19 stream-collide kernels (Eq. 22-28).
#pragma once
#include "common.cuh"

// Eq. (22a), (22b): density and velocity of one cell.  Opposite directions are paired (q, q+1), so the sums
// are short trees rather than 19-long dependent chains.
template <typename T>
__device__ __forceinline__ void lb_moments(const T (&f)[LEDDS_Q], T& rho, T& ux, T& uy, T& uz)
{
    T s[9], d[9];
#pragma unroll
    for (int p = 0; p < 9; ++p) { s[p] = f[2 * p + 1] + f[2 * p + 2]; d[p] = f[2 * p + 1] - f[2 * p + 2]; }
    const T r = (f[0] + s[0]) + ((s[1] + s[2]) + (s[3] + s[4])) + ((s[5] + s[6]) + (s[7] + s[8]));
    T jx = T(0), jy = T(0), jz = T(0);
#pragma unroll
    for (int p = 0; p < 9; ++p) {                         // d[p] = f_q - f_opp(q) carries c_q
        const int q = 2 * p + 1;
        if (lb_cx(q) == 1) jx += d[p]; else if (lb_cx(q) == -1) jx -= d[p];
        if (lb_cy(q) == 1) jy += d[p]; else if (lb_cy(q) == -1) jy -= d[p];
        if (lb_cz(q) == 1) jz += d[p]; else if (lb_cz(q) == -1) jz -= d[p];
    }
    const T inv = T(1) / r;
    rho = r; ux = jx * inv; uy = jy * inv; uz = jz * inv;
}

// c_q . u with the zero components folded away at compile time.
template <typename T>
__device__ __forceinline__ T lb_cdot(int q, T ux, T uy, T uz)
{
    T s = T(0);
    if (lb_cx(q) == 1) s += ux; else if (lb_cx(q) == -1) s -= ux;
    if (lb_cy(q) == 1) s += uy; else if (lb_cy(q) == -1) s -= uy;
    if (lb_cz(q) == 1) s += uz; else if (lb_cz(q) == -1) s -= uz;
    return s;
}

// Eq. (28) with c_s^2 = 1/3 for all 19 directions.
template <typename T>
__device__ __forceinline__ void lb_equilibrium(T (&fe)[LEDDS_Q], T rho, T ux, T uy, T uz)
{
    const T k = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    fe[0] = T(lb_w(0)) * rho * k;
#pragma unroll
    for (int q = 1; q < LEDDS_Q; q += 2) {            // q and q+1 are opposites
        const T cu = lb_cdot(q, ux, uy, uz);
        const T wr = T(lb_w(q)) * rho;
        const T even = wr * (k + T(4.5) * cu * cu), odd = wr * T(3) * cu;
        fe[q] = even + odd;
        fe[q + 1] = even - odd;
    }
}

// Eq. (24), (26): f* = f - omega (f - feq), in place.
template <typename T>
__device__ __forceinline__ void lb_collide_bgk(T (&f)[LEDDS_Q], T omega, T rho, T ux, T uy, T uz)
{
    T fe[LEDDS_Q];
    lb_equilibrium(fe, rho, ux, uy, uz);
#pragma unroll
    for (int q = 0; q < LEDDS_Q; ++q) f[q] = f[q] - omega * (f[q] - fe[q]);
}

// Eq. (29)-(30): TRT.  f+- = (f_q +- f_qbar)/2 relax with dt/tau+ and dt/tau- towards the even and odd parts
// of the equilibrium; the rest population has no odd part.
template <typename T>
__device__ __forceinline__ void lb_collide_trt(T (&f)[LEDDS_Q], T omega_p, T omega_m, T rho, T ux,
                                               T uy, T uz)
{
    const T k = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    f[0] = f[0] - omega_p * (f[0] - T(lb_w(0)) * rho * k);
#pragma unroll
    for (int q = 1; q < LEDDS_Q; q += 2) {
        const T cu = lb_cdot(q, ux, uy, uz);
        const T wr = T(lb_w(q)) * rho;
        const T even = wr * (k + T(4.5) * cu * cu), odd = wr * T(3) * cu;
        const T rp = omega_p * (T(0.5) * (f[q] + f[q + 1]) - even), rm = omega_m * (T(0.5) * (f[q] - f[q + 1]) - odd);
        f[q] = f[q] - (rp + rm);
        f[q + 1] = f[q + 1] - (rp - rm);
    }
}

// the collision model is a compile-time choice: each kernel is instantiated for BGK and for TRT
template <bool TRT, typename T>
__device__ __forceinline__ void lb_collide(T (&f)[LEDDS_Q], const LbmDev& P, T rho, T ux, T uy, T uz)
{
    if (TRT) lb_collide_trt(f, (T)P.omega, (T)P.omega_minus, rho, ux, uy, uz);
    else lb_collide_bgk(f, (T)P.omega, rho, ux, uy, uz);
}

// cells along x covered by one 128-thread block (the rest of the block goes along y)
static inline int lb_block_x(int nx) { return nx > 64 ? 128 : (nx > 32 ? 64 : 32); }

// Index type of the population arrays: unsigned 32-bit when 19 N < 2^32 (one IMAD.WIDE per access), else 64-bit.
static inline bool lb_fits_u32(long long N) { return (unsigned long long)N * LEDDS_Q < 0xffffffffull; }

// The 19 pre-collision populations of cell `cell`.
template <typename I, typename T>
__device__ __forceinline__ void lb_load(const T* __restrict__ fin, I N, I cell, T (&f)[LEDDS_Q])
{
#pragma unroll
    for (int q = 0; q < LEDDS_Q; ++q) f[q] = __ldg(fin + (I)((I)q * N + cell));
}

// Eq. (25) as a push of the post-collision populations of cell (x,y,z), with boundaries.
// The neighbour coordinates and "this link leaves through a wall" flags are worked out once per axis and
// the nine row offsets once per block (y and z are uniform over the block), so a direction costs a
// predicate, an index and a store.
template <typename I>
struct LbPush {
    int x, tx[3];                 // tx[0] / tx[2]: target x for c_x = -1 / +1
    unsigned wmask;               // bit 2 a + s: a link towards side s (0 low, 1 high) of axis a leaves through a wall
    I N, rb[3][3];                // row offsets [c_z + 1][c_y + 1]

    __device__ __forceinline__ LbPush(const LbmDev& P, int x_, int y, int z) : x(x_), wmask(0u), N((I)P.N)
    {
        int ty[3] = {y - 1, y, y + 1}, tz[3] = {z - 1, z, z + 1};
        tx[0] = x - 1; tx[1] = x; tx[2] = x + 1;
        if (x == 0) { if (P.bc[0]) wmask |= 1u; else tx[0] = P.nx - 1; }
        if (x == P.nx - 1) { if (P.bc[0]) wmask |= 2u; else tx[2] = 0; }
        if (y == 0) { if (P.bc[1]) wmask |= 4u; else ty[0] = P.ny - 1; }
        if (y == P.ny - 1) { if (P.bc[1]) wmask |= 8u; else ty[2] = 0; }
        if (z == 0) { if (P.bc[2]) wmask |= 16u; else tz[0] = P.nz - 1; }
        if (z == P.nz - 1) { if (P.bc[2]) wmask |= 32u; else tz[2] = 0; }
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) rb[a][b] = ((I)tz[a] * (I)P.ny + (I)ty[b]) * (I)P.nx;
    }

    // walls a link of direction q can leave through (compile-time constant after unrolling)
    static __device__ __forceinline__ constexpr unsigned link_mask(int q)
    {
        return (lb_cx(q) < 0 ? 1u : (lb_cx(q) > 0 ? 2u : 0u)) | (lb_cy(q) < 0 ? 4u : (lb_cy(q) > 0 ? 8u : 0u)) |
               (lb_cz(q) < 0 ? 16u : (lb_cz(q) > 0 ? 32u : 0u));
    }

    // post-collision population v of direction q (a compile-time constant after unrolling); rho = the cell's
    // pre-collision density (moving-wall term, G19).  A cell away from every wall (wmask == 0: all but the outermost
    // layer of a walled axis) takes the first branch for all 19 directions: an index and a store.
    // NOWALL: the caller has found wmask == 0 for every lane of the warp: no test
    template <typename T, bool NOWALL = false>
    __device__ __forceinline__ void put(T* __restrict__ fout, const LbmDev& P, int q, T v, T rho) const
    {
        const int cx = lb_cx(q), cy = lb_cy(q), cz = lb_cz(q);
        if (NOWALL || (wmask & link_mask(q)) == 0u) {
            fout[(I)((I)q * N + rb[cz + 1][cy + 1] + (I)tx[cx + 1])] = v;
        } else {
            T cuw = T(0);                                   // c_q . u_wall summed over the crossed walls
            if (P.any_wall_velocity) {
                if (cx != 0 && (wmask & (cx > 0 ? 2u : 1u))) { const double* uw = P.uw + (0 + (cx > 0)) * 3; cuw += lb_cdot(q, (T)uw[0], (T)uw[1], (T)uw[2]); }
                if (cy != 0 && (wmask & (cy > 0 ? 8u : 4u))) { const double* uw = P.uw + (2 + (cy > 0)) * 3; cuw += lb_cdot(q, (T)uw[0], (T)uw[1], (T)uw[2]); }
                if (cz != 0 && (wmask & (cz > 0 ? 32u : 16u))) { const double* uw = P.uw + (4 + (cz > 0)) * 3; cuw += lb_cdot(q, (T)uw[0], (T)uw[1], (T)uw[2]); }
            }
            fout[(I)((I)lb_opp(q) * N + rb[1][1] + (I)x)] = v - T(6.0 * lb_w(q)) * rho * cuw;
        }
    }
};

template <typename I, typename T>
__device__ __forceinline__ void lb_push_store(T* __restrict__ fout, const LbmDev& P, int x, int y, int z,
                                              const T (&fs)[LEDDS_Q], T rho)
{
    const LbPush<I> push(P, x, y, z);
#pragma unroll
    for (int q = 0; q < LEDDS_Q; ++q) push.put(fout, P, q, fs[q], rho);
}
