// common.cuh -- shared device-side types of the DD-4DVar CUDA path (sm_100a).
// Product code: shares nothing with oracle/.  Citations "l.N" are PAPER.md lines.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define DD_NF 3      // fields h,u,v
#define DD_GHOST 3   // stencil reach of one full step: stage A 1 + h1 1 + u1/v1 1 (R14)

// One space-time subdomain Delta_j x Omega_i (Def 3 l.128-154) as the kernels see it.
struct Sub {
    int a, b, jw;            // tile column, tile row, window
    int ei0, ej0, ex, ey;    // extended tile: origin (column unwrapped, may be < 0), size (eq (70) l.1024)
    int gx, gys, gyn;        // ghost widths: 0 = side closed by the model's own rule
    int px, py;              // padded tile = extended tile + ghost ring
    int s, W;                // first time level, number of model steps in the window
    int ncell, npad, nring;  // ex*ey, px*py, npad - ncell
    int oi0, oi1, oj0, oj1;  // owned ranges
    long long coff;          // offset (doubles) in control-shaped arrays [3][ncell]
    long long toff;          // offset in the trajectory store [(W+1)][3][ncell]
    long long goff;          // offset in the ghost store [W][3][nring]
    long long poff;          // offset in padded scratch arrays [3][npad] (single-field: poff/3)
    long long ooff;          // index into obs_start: entries ooff .. ooff+W+1
    long long eoff;          // offset in the edge store [W][py][2] (frozen u^a of ghost columns 1, px-2)
    int nb0, nnb;            // this subdomain's overlap rectangles: entries nb0 .. nb0+nnb-1 of the NbRect table
    int novl;                // cells of all those rectangles together
    long long voff;          // offset in the overlap store [W][3][novl] (levels 1 .. W; option overlap_levels)
};

// One rectangle Omega_i ∩ Omega_k of the spatial overlap (eq (20)-(22) l.294-306, case 1 l.310-314):
// cells (i0 + di, j0 + dj) of this tile coincide with cells (ni0 + di, nj0 + dj) of the
// neighbour tile in the same window, whose control starts at coff2 (shape [3][ncell2], row length ex2).
struct NbRect {
    long long coff2;
    long long toff2;         // the neighbour's offset in the trajectory store
    int ex2, ncell2, i0, j0, w, h, ni0, nj0;
    int ooff;                // first cell of this rectangle in the subdomain's overlap list (row-major inside the rectangle)
};

// Model constants with dt folded in (row tables live in device memory, length nlat).
struct ModelP {
    int nlon, nlat;
    double kap;              // index-space diffusion kappa (R3)
    double dtcm;             // dt / (2 a dtheta)
    double gdtcm;            // g dt / (2 a dtheta)
    const double* dtcz;      // dt / (2 a dlambda m_j)
    const double* gdtcz;     // g dt / (2 a dlambda m_j)
    const double* dtf;       // dt 2 Omega sin(theta_j)
    const double* dtt;       // dt sin(theta_j) / (a m_j)
    const double* rp;        // m_{j+1}/m_j
    const double* rm;        // m_{j-1}/m_j
};

// Geometry tables of one layout (device pointers).
struct GeoP {
    int nlon, nlat, p1, p2, q;
    const int* colown;   // [nlon] owner tile column
    const int* rowown;   // [nlat]
    const int* ncolcov;  // [nlon] number of tile columns whose extended range covers the column
    const int* colcov;   // [4*nlon]
    const int* nrowcov;  // [nlat]
    const int* rowcov;   // [4*nlat]
    const int* tc_ei0;   // [p1] extended origin of tile column a
    const int* tc_ex;    // [p1]
    const int* tr_ej0;   // [p2]
    const int* tr_ey;    // [p2]
    const int* wb;       // [q+1] window boundaries
};

// Statistics and weights of the functional, eq (6) l.111 and eq (25) l.338-344.
struct CostP {
    double ib[3];        // 1 / sigma_b^2 per field
    double sb[3];        // sigma_b
    double mu, lambda;
    double bgw;          // weight of (25a) in the windows j > 0 (R7): 0 = only at t_0, 1 = as printed
};

__device__ __forceinline__ int imodd(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

// Deterministic block-wide sum (fixed tree: lane shuffles, then warp partials in order).
template <int NT>
__device__ __forceinline__ double block_sum(double v, double* sh /*[32]*/)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = lane < (NT >> 5) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
        if (lane == 0) sh[0] = r;
    }
    __syncthreads();
    r = sh[0];
    return r;
}
template <int NT>
__device__ __forceinline__ double block_max(double v, double* sh)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = lane < (NT >> 5) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r = fmax(r, __shfl_down_sync(0xffffffffu, r, o));
        if (lane == 0) sh[0] = r;
    }
    __syncthreads();
    r = sh[0];
    return r;
}
