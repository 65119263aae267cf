// wave_common.cuh -- shared pieces of the WAVEFRONT sweep kernels (wave_forward.cuh, wave_adjoint.cuh).
//
// Design ("smem-resident tile, temporal wavefront").  One CTA of WK_NW warps works
// through the space-time subdomains Delta_j x Omega_i (Def 3 l.128-154) blockIdx.x, blockIdx.x + gridDim.x,
// ... as ONE continuous pipeline of model steps: the first step of a subdomain follows the last step of the
// previous one row by row, like any other step (no CTA-wide phase, no __syncthreads after start-up; the
// control-level terms of J_ji run in the bandwidth-bound kernel ck_cost).  The state of the window
// (forward: Z^n, adjoint: the adjoint variable lambda^n and u^n) lives IN PLACE in shared memory for
// the whole window.  Warp w works on a DIFFERENT TIME STEP than its neighbours: it marches over the
// rows of the tile a few rows behind the warp that produces its input level (its "leader") and a
// few rows ahead of the warp that consumes its output (its "follower").  All sub-stages of one
// model step (R3) run software-pipelined on different rows inside one warp, so
//   - north/south neighbours are the lane's own registers (row history),
//   - east/west neighbours are the lane's own registers or ONE warp shuffle per K columns
//     (every lane owns K adjacent columns; a warp spans the whole tile width),
//   - there is no __syncthreads and no shared-memory exchange inside a step: the only
//     inter-warp communication is the state row itself plus a progress word (release/acquire),
//   - HBM sees exactly the algorithmic traffic: trajectory rows leave (forward) or arrive (adjoint)
//     through TMA bulk copies (cp.async.bulk + mbarrier), the frozen ghost ring arrives the same
//     way; nothing is staged through registers, nothing is re-read.
// Eligibility (host, wave_plan): every tile has a ghost ring in longitude (p_lon >= 2), an even
// number of columns (16-byte aligned rows for the bulk copies), at most 32 K + 4 padded columns
// (K = 2 or 3 columns per lane) and the shared-memory layout fits in 227 KB.  Other layouts run
// the row-marching kernels (fused_kernels.cuh) or the generic kernels.
#pragma once
#include <stdint.h>
#include "common.cuh"
#include "model_math.cuh"

#ifndef WK_NW
#define WK_NW 8                 // warps per CTA = time steps in flight per CTA
#endif
#define WK_NT (WK_NW * 32)
#define WK_EWC 4                // tile rows per staged chunk of east/west ghost cells (forward kernel)
#define WK_EWCA 2               // the same in the adjoint kernel (its shared memory is full)
#define WK_HDR 128              // doubles reserved at the start of shared memory (barriers, flags)
#define WK_NTAB 3               // row-table slots: 8 steps in flight span at most 3 subdomains when every window has >= 4 steps
#define WK_TABSZ(maxpy) (((maxpy) + 2) * 8)
#define WK_SMEM_MAX 232448      // 227 KB: largest opt-in dynamic shared memory of one CTA on sm_100a
// Adjoint kernel: the strides of its shared-memory arrays are COMPILE-TIME constants of K (immediate offsets in the
// hot loop instead of address arithmetic): ring row pitch 32 K + 6 (the widest padded row + 2), lambda / u^n field
// stride (WK_AROWS + 1) rows of 32 K cells, WK_AROWS = the tallest extended tile the 227 KB hold.
#define WK_AZP(K) (32 * (K) + 6)
#define WK_AROWS(K) ((K) == 3 ? 49 : 80)
#define WK_AFS(K) ((WK_AROWS(K) + 1) * 32 * (K))

// Shared-memory layout in doubles (same function on host and device).
//   header | row tables [WK_NTAB][(maxpy+2)][8] | resident state | per-warp staging
// forward resident state: [3][WK_AROWS][P] with pitch P = WK_AZP = 32 K + 6 >= maxex + 8; a tile row holds
//   [tile ex][E ghosts 3][pad 2][W ghosts of the NEXT row 3], so that padded column c of tile row
//   lj is at  st + f*FS + lj*P + (c - 3)  for every c (W ghosts sit in the previous row's tail).
// adjoint resident state: lambda [3][WK_AROWS+1][32 K] and u1 [WK_AROWS+1][32 K]: lambda is zero outside
//   the extended tile, so only the columns the lanes own are kept; the cells of ghost columns and
//   the extra row stay zero and serve every read that falls outside the tile.
struct WkLayout {
    int tab, st, P, FS, u1, wbase, wsz, sn, zr, ZP, ew, eds, ede, total;
};
__host__ __device__ inline WkLayout wk_layout(bool adj, int maxex, int maxey, int maxpx, int maxpy)
{
    WkLayout L;
    int o = WK_HDR;
    L.tab = o; o += WK_NTAB * WK_TABSZ(maxpy);      // row tables of the subdomains in flight
    if (!adj) {
        L.P = WK_AZP(maxpx - 4 <= 64 ? 2 : 3); L.FS = WK_AROWS(maxpx - 4 <= 64 ? 2 : 3) * L.P;    // (compile-time in the kernel)
        L.st = o + 8; o += 8 + 3 * L.FS + 64;       // 64 doubles of slack: lanes beyond px read past a row
        L.u1 = 0;
    } else {
        // row pitch = 32 K cells (one cell per lane and owned column: cell q <-> padded column q + 2, so
        // q = 0 and q > ex are permanently zero), plus one all-zero row (index maxey) per field
        // (field stride and ring pitch do not depend on the layout: WK_AFS, WK_AZP; row WK_AROWS is the all-zero row)
        const int K = maxpx - 4 <= 64 ? 2 : 3;
        L.P = 32 * K; L.FS = WK_AFS(K);
        L.st = o; o += 3 * L.FS;
        L.u1 = o; o += L.FS;
    }
    L.wbase = o;
    int p = 0;
    L.ZP = adj ? WK_AZP(maxpx - 4 <= 64 ? 2 : 3) : maxpx + 2;
    if (!adj) { L.sn = p; p += 9 * maxpx; L.zr = 0; }
    else { L.zr = p; p += 9 * L.ZP; L.sn = 0; }
    const int ewc = adj ? WK_EWCA : WK_EWC;
    L.ew = p; p += 2 * 3 * 6 * ewc;
    L.eds = p; p += 16;
    L.ede = p; p += 2 * 2 * ewc;
    L.wsz = (p + 1) & ~1;
    L.total = L.wbase + WK_NW * L.wsz + 64;
    return L;
}

// Kernel arguments (by value; everything the two kernels need).
struct WkArgs {
    const Sub* subs; const NbRect* nbr; const int* mask; int nsub; int* counter;
    ModelP m; CostP cp; GeoP geo;
    const double *x, *xbs, *xfrozen, *pred_end;
    double* traj; const double* ghost; const double* gedge;
    const long long* obs_start; const int* obs_idx; const int* obs_lj;
    const double *obs_y, *obs_c; double* obs_r;
    double *parts, *J;          // forward outputs: [nsub][5], [nsub]
    double *gx, *gw;            // adjoint outputs
    int maxex, maxey, maxpx, maxpy;
    const double* wtab; int wtab_stride;    // row tables per tile row b: [p2][maxpy + 2][8] (entry r+1 <-> padded row r = -1 .. py)
    double* lamW;               // [ctot] adjoint variable at the window end, written by ck_cost: 2 mu (Z^W - x_succ) / sigma_b^2
    WkLayout Lf, La;            // shared-memory layouts (forward, adjoint), computed on the host: constant-bank operands
};

// ------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier, TMA bulk copies (cp.async.bulk), proxy fence, release/acquire flags.
__device__ __forceinline__ uint32_t wk_s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void wk_mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(wk_s32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void wk_mbar_expect(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(wk_s32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool wk_mbar_try(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(wk_s32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void wk_mbar_wait(uint64_t* bar, uint32_t parity)
{
    while (!wk_mbar_try(bar, parity)) {}
}
// global -> shared bulk copy; completion is signalled on `bar` (complete_tx); 16-byte aligned
__device__ __forceinline__ void wk_g2s(double* dst, const double* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(wk_s32(dst)), "l"(src), "r"(bytes), "r"(wk_s32(bar)) : "memory");
}
// shared -> global bulk copy (bulk async-group)
__device__ __forceinline__ void wk_s2g(double* dst, const double* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(dst), "r"(wk_s32(src)), "r"(bytes) : "memory");
}
// the same with 32-bit shared-window addresses (no generic-to-shared conversion in the hot loop)
__device__ __forceinline__ void wk_mbar_init32(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void wk_mbar_expect32(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void wk_mbar_wait32(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void wk_g2s32(uint32_t dst, const double* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void wk_s2g32(double* dst, uint32_t src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void wk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void wk_wait_read()
{
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
// generic-proxy writes to shared memory -> visible to the async proxy (TMA store source)
__device__ __forceinline__ void wk_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void wk_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// Progress words.  Writer: every lane stores its cells of the row (st.shared), __syncwarp, then ONE lane stores
// the word with release semantics; reader: polls the word with acquire semantics, then loads the row.  The pair
// st.release.cta / ld.acquire.cta is what the PTX memory model asks for between the row data (weak accesses) and the
// word; it costs one MEMBAR.ALL.CTA per tick on either side (about 1 % of the sweep against plain volatile accesses,
// DESIGN.md section 5), which is the price of not resting the hot path on the issue order of one SM's shared-memory pipe.
__device__ __forceinline__ void wk_publish(uint32_t addr, unsigned v)
{
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned wk_peek(uint32_t addr)
{
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
#define WK_BACKOFF __nanosleep(40)
// wait until the progress word at `addr` has reached `need` (monotone counters, wrap-safe compare)
__device__ __forceinline__ void wk_wait_prog(uint32_t addr, unsigned need)
{
    while ((int)(wk_peek(addr) - need) < 0) { WK_BACKOFF; }
}

// ------------------------------------------------------------------------------------------
// Per-subdomain geometry as a warp sees it (uniform over the CTA).
struct WkGeo {
    int ex, ey, px, py, gys, gyn, ncell, nring, W, joff;
    bool ws, wn;            // pole walls (R4)
};
__device__ __forceinline__ WkGeo wk_geo(const Sub& s)
{
    WkGeo g;
    g.ex = s.ex; g.ey = s.ey; g.px = s.px; g.py = s.py; g.gys = s.gys; g.gyn = s.gyn;
    g.ncell = s.ncell; g.nring = s.nring; g.W = s.W; g.joff = s.ej0 - s.gys;
    g.ws = s.gys == 0; g.wn = s.gyn == 0;
    return g;
}
// Row tables (host-built, dd4dvar.cu): entry r+1 for padded row r = -1 .. py of a tile row, with the guard
// values r+_{-1} = 1 and r-_{nlat} = 1 of the virtual mirrored pole rows (model_math.cuh, A_v).  The warp
// that runs the first step of a subdomain copies the table of its tile row into slot (ordinal % WK_NTAB)
// before its first tick; the steps behind it see it through the progress words.
__device__ __forceinline__ void wk_copy_tab(double* dst, const double* __restrict__ src, int py, int lane)
{
    for (int q = lane; q < (py + 2) * 8; q += 32) dst[q] = __ldg(src + q);
}
#define WK_T_DTCZ 0
#define WK_T_GDTCZ 1
#define WK_T_DTF 2
#define WK_T_DTT 3
#define WK_T_RP 4
#define WK_T_RM 5
#define WK_T_CMRP 6             // dtcm * r+
#define WK_T_CMRM 7             // dtcm * r-
#define WK_BAR_PER_WARP 8       // mbarriers per warp at the start of shared memory
#define WK_PROG 64              // progress words (one u32 per warp) at double index WK_PROG

// Position of a physical warp in the step order: the identity.  (Warps p and p + 4 share a scheduler; other distances of
// such a pair in the step order were measured and bought nothing, profiles/r2_wave_v2.md.)
__device__ __forceinline__ int wk_logical_warp(int p) { return p; }

// one elected lane of the (converged) warp; tells the compiler the region is single-threaded
__device__ __forceinline__ bool wk_elect()
{
    uint32_t p;
    asm volatile("{\n\t.reg .pred q;\n\telect.sync _|q, 0xffffffff;\n\tselp.u32 %0, 1, 0, q;\n\t}" : "=r"(p));
    return p != 0;
}
// broadcast from lane 0: marks a value as warp-uniform for the compiler (uniform datapath, no vote loops)
__device__ __forceinline__ int wk_uni(int v) { return __shfl_sync(0xffffffffu, v, 0); }

// shared-memory access with an explicit 32-bit shared-window address and a compile-time byte offset
// (the steady ticks keep running addresses in registers; volatile: program order is the schedule)
template <int OFF> __device__ __forceinline__ double wk_lds(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(a), "n"(OFF) : "memory");
    return v;
}
template <int OFF> __device__ __forceinline__ void wk_sts(uint32_t a, double v)
{
    asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(a), "n"(OFF), "d"(v) : "memory");
}

// 8-byte asynchronous copy global -> shared by every lane (LDGSTS), per-thread groups
__device__ __forceinline__ void wk_cpa8(uint32_t dst, const double* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void wk_cpa_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void wk_cpa_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// 64-bit shuffles
__device__ __forceinline__ double wk_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double wk_dn(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
