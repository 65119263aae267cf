// fused_kernels.cuh -- the fused persistent sweep kernels (fused_forward.cuh, fused_adjoint.cuh):
// a CTA of 128 threads takes subdomains from a work counter and runs the whole window of each one
// (forward: all W steps; adjoint: all W steps backwards) without leaving the kernel.
//
// Design ("row marching"): thread i owns padded column i of the tile
// and marches over the rows.  All sub-stages of a step run software-pipelined on different rows
// in the same tick, so one __syncthreads per row:
//   forward  tick t : load Z0[t] | stage A row t-1 | h1 row t-2 | u1,v1 row t-3 -> store
//   adjoint  tick t : load Z0[t] | stage A row t-1, UB row t-1 | HB,P row t-2 | A row t-3 |
//                     lam0 row t-4 -> store
// North/south neighbours are the thread's own registers (static slots, row & 3); east/west
// neighbours come from small shared-memory row rings written one tick earlier; row tables sit in
// constant memory.  HBM sees each trajectory level once per sweep direction (streaming write in
// the forward kernel, read in the adjoint kernel) plus the frozen ghost ring.  The forward state
// and the adjoint variable are updated IN PLACE (row j rewritten 3-4 ticks after the same thread
// read it) in a per-CTA slot of a scratch that is pinned in L2 (access-policy window).
// No step is recomputed except stage A in the adjoint, no atomics on data: deterministic results.
#pragma once
#include <stdlib.h>
#include <string.h>
#include "common.cuh"
#include "model_math.cuh"

#define FK_MAXNT 128       // widest padded tile the fused kernels take (threads per CTA: 64 or 128)
#define FK_ZR 8            // depth of the Z0 row ring (adjoint reads rows t-5 .. t)

struct FusedPlan {
    int enabled = 0;
    // what fused_setup changed and fused_teardown puts back (device limit, stream attribute)
    bool l2_set = false;
    size_t l2_prev_limit = 0;
    cudaStreamAttrValue l2_prev_attr;
    int maxpy = 0, maxncell = 0;
    size_t smem_fwd = 0, smem_adj = 0;
    // persistent CTAs: one L2-persistent scratch slot per resident CTA (in-place state / adjoint variable)
    int nt = 128;                     // threads per CTA (64 for narrow tiles)
    int nslots = 0, nslots_fwd = 0;
    long long slot_stride = 0;        // doubles
    double* scratch = nullptr;
    int* counter = nullptr;
};
#define FK_SMS 148                  // B200
#define FK_ADJ_CTAS 3                // resident adjoint CTAs per SM at 128 threads (register budget 168)
typedef void* (*fused_take_fn)(void* arena, size_t bytes);

inline bool fused_fits(const Sub* subs, int nsub)
{
    for (int k = 0; k < nsub; ++k)
        if (subs[k].px > FK_MAXNT || subs[k].py < 1) return false;
    return nsub > 0;
}
inline void fused_plan_init(FusedPlan& fp, const Sub* subs, int nsub, int lam_mode);
inline void fused_plan_arrays(FusedPlan& fp, fused_take_fn take, void* arena)
{
    if (!fp.enabled) return;
    fp.scratch = (double*)take(arena, sizeof(double) * (size_t)fp.nslots_fwd * fp.slot_stride);
    fp.counter = (int*)take(arena, 64);
}

// ------------------------------------------------------------------------------------------
// Per-thread view of the marching CTA.  Row conditions are uniform over the CTA (plain branches);
// column conditions are per-thread constants.  Values computed outside a stage's valid range are
// finite and are never consumed by a valid cell, so only the adjoint
// variable (zero outside the extended tile) and the global stores are predicated per thread.
struct FkGeo {
    int px, py, ex, ey, gx, gys, gyn, joff, ncell, nring;
    bool perx, ws, wn;
    int i, li, iE, iW;
    bool col_ok, cU;
    int jA0, jA1, jH0, jH1, jU0, jU1;     // row ranges of stage A / h1 / u1,v1 (half open)
};
__device__ __forceinline__ FkGeo fk_geo(const Sub& s)
{
    FkGeo g;
    g.px = s.px; g.py = s.py; g.ex = s.ex; g.ey = s.ey; g.gx = s.gx; g.gys = s.gys; g.gyn = s.gyn;
    g.joff = s.ej0 - s.gys; g.ncell = s.ncell; g.nring = s.nring;
    g.perx = s.gx == 0; g.ws = s.gys == 0; g.wn = s.gyn == 0;
    g.i = threadIdx.x; g.li = g.i - s.gx;
    g.col_ok = g.i < s.px;
    g.iE = g.i + 1 < s.px ? g.i + 1 : (g.perx ? 0 : g.i);
    g.iW = g.i > 0 ? g.i - 1 : (g.perx ? s.px - 1 : 0);
    if (!g.col_ok) { g.iE = g.iW = g.i; }
    g.cU = g.col_ok && g.li >= 0 && g.li < s.ex;
    g.jA0 = g.ws ? 0 : 1; g.jA1 = g.wn ? s.py : s.py - 1;
    g.jH0 = g.ws ? 0 : 2; g.jH1 = g.wn ? s.py : s.py - 2;
    g.jU0 = s.gys; g.jU1 = s.gys + s.ey;
    return g;
}

// where this thread's column of the padded rows of one level lives: south ghost rows, tile rows
// (trajectory store for tile columns, ghost strip otherwise), north ghost rows
struct FkCol {
    const double *pS, *pI, *pN;
    int sI;
    long long fI, fG;
};
__device__ __forceinline__ FkCol fk_col(const FkGeo& g, const double* tz, const double* gz)
{
    FkCol c;
    const int i = g.col_ok ? g.i : 0;
    c.fG = g.nring;
    c.pS = gz + i;
    c.pN = gz + g.gys * g.px + i;
    if (g.cU || !g.col_ok) { c.pI = tz + (g.col_ok ? g.li : 0); c.sI = g.ex; c.fI = g.ncell; }
    else { c.pI = gz + (g.gys + g.gyn) * g.px + (i < g.gx ? i : i - g.ex); c.sI = 2 * g.gx; c.fI = g.nring; }
    return c;
}
__device__ __forceinline__ void fk_load_row(const FkGeo& g, const FkCol& c, int j, double z[3])
{
    const double* p; long long fs;
    if (j < g.gys) { p = c.pS + j * g.px; fs = c.fG; }
    else if (j < g.gys + g.ey) { p = c.pI + (j - g.gys) * c.sI; fs = c.fI; }
    else { p = c.pN + (j - g.gys - g.ey) * g.px; fs = c.fG; }
    z[0] = p[0]; z[1] = p[fs]; z[2] = p[2 * fs];
}

// Row tables of the static-slot kernels: entry [k][gj + 1], with guard entries r+_{-1} = 1 and
// r-_{nlat} = 1 for the virtual mirrored pole rows.  They live in a per-HANDLE device buffer (no
// process-global state: two handles on two streams never share tables) and are read with uniform
// (per-CTA) indices through the read-only path; `C.tb` is the tick context's pointer to them.
#define FK_CTAB 1026
#define CT_DTCZ 0
#define CT_GDTCZ 1
#define CT_DTF 2
#define CT_DTT 3
#define CT_RP 4
#define CT_RM 5
#define ctab(k, cj, j) __ldg(C.tb + (k) * FK_CTAB + (cj) + (j))

// the kernels are instantiated for CTAs of 128 threads (tiles up to 128 padded columns) and of 64
// threads (narrow tiles, e.g. the 16x16x8 layout of config 4: 55 columns)
#define FK_NT 128
namespace fk128 {
#include "fused_adjoint.cuh"
#include "fused_forward.cuh"
}
#undef FK_NT
#define FK_NT 64
namespace fk64 {
#include "fused_adjoint.cuh"
#include "fused_forward.cuh"
}
#undef FK_NT

inline void fused_plan_init(FusedPlan& fp, const Sub* subs, int nsub, int lam_mode)
{
    fp = FusedPlan();
    if (!subs || nsub <= 0) return;
    fp.enabled = 1;
    for (int k = 0; k < nsub; ++k) {
        fp.maxpy = subs[k].py > fp.maxpy ? subs[k].py : fp.maxpy;
        fp.maxncell = subs[k].ncell > fp.maxncell ? subs[k].ncell : fp.maxncell;
    }
    int maxpx = 0;
    for (int k = 0; k < nsub; ++k) maxpx = subs[k].px > maxpx ? subs[k].px : maxpx;
    fp.nt = maxpx <= 64 ? 64 : 128;
    const int sa = FK_SMS * (FK_ADJ_CTAS * 128 / fp.nt), sf = FK_SMS * (512 / fp.nt);   // resident CTAs: adjoint, forward
    fp.nslots = nsub < sa ? nsub : sa;
    fp.nslots_fwd = nsub < sf ? nsub : sf;
    fp.slot_stride = (3LL * fp.maxncell + 31) & ~31LL;
    fp.smem_fwd = 0;
    fp.smem_adj = 0;
}
// copy the row tables (host, 6 x nlat, order dtcz gdtcz dtf dtt rp rm) into this handle's device buffer
// d_ctab [6][FK_CTAB]; `stage` (host, same size, owned by the handle) must outlive the async copy
inline int fused_upload_tables(cudaStream_t stream, const double* h_tab, int nlat, double* stage, double* d_ctab)
{
    if (nlat + 2 > FK_CTAB) return -1;
    for (int k = 0; k < 6; ++k) {
        double* b = stage + (size_t)k * FK_CTAB;
        for (int q = 0; q < FK_CTAB; ++q) b[q] = 0.0;
        for (int j = 0; j < nlat; ++j) b[j + 1] = h_tab[(size_t)k * nlat + j];
        b[0] = b[1]; b[nlat + 1] = b[nlat];
    }
    stage[(size_t)CT_RP * FK_CTAB] = 1.0; stage[(size_t)CT_RM * FK_CTAB + nlat + 1] = 1.0;
    return cudaMemcpyAsync(d_ctab, stage, sizeof(double) * 6 * FK_CTAB, cudaMemcpyHostToDevice, stream) == cudaSuccess ? 0 : -1;
}
inline int fused_setup(cudaStream_t stream, FusedPlan& fp, const Sub*)
{
    if (!fp.enabled) return 0;
    {   // keep the per-CTA scratch resident in L2; everything else streams through the rest
        int dev = 0; cudaGetDevice(&dev);
        cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
        size_t bytes = sizeof(double) * (size_t)fp.nslots_fwd * fp.slot_stride;
        size_t lim = bytes < (size_t)prop.persistingL2CacheMaxSize ? bytes : (size_t)prop.persistingL2CacheMaxSize;
        if (lim > 0) {
            memset(&fp.l2_prev_attr, 0, sizeof(fp.l2_prev_attr));
            cudaDeviceGetLimit(&fp.l2_prev_limit, cudaLimitPersistingL2CacheSize);
            cudaStreamGetAttribute(stream, cudaStreamAttributeAccessPolicyWindow, &fp.l2_prev_attr);
            fp.l2_set = true;
            if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, lim > fp.l2_prev_limit ? lim : fp.l2_prev_limit) != cudaSuccess) return -1;
            cudaStreamAttrValue av; memset(&av, 0, sizeof(av));
            av.accessPolicyWindow.base_ptr = fp.scratch;
            av.accessPolicyWindow.num_bytes = bytes < (size_t)prop.accessPolicyMaxWindowSize ? bytes : (size_t)prop.accessPolicyMaxWindowSize;
            av.accessPolicyWindow.hitRatio = lim >= bytes ? 1.0f : (float)lim / (float)bytes;
            av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
            av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
            if (cudaStreamSetAttribute(stream, cudaStreamAttributeAccessPolicyWindow, &av) != cudaSuccess) return -1;
        }
    }
    return 0;
}
// undo fused_setup: the stream gets its previous access-policy window back, persisting lines are
// released, the device-wide persisting-L2 limit returns to what it was
inline void fused_teardown(cudaStream_t stream, FusedPlan& fp)
{
    if (!fp.l2_set) return;
    cudaStreamSynchronize(stream);
    cudaStreamSetAttribute(stream, cudaStreamAttributeAccessPolicyWindow, &fp.l2_prev_attr);
    cudaCtxResetPersistingL2Cache();
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, fp.l2_prev_limit);
    fp.l2_set = false;
}
