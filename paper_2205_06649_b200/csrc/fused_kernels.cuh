// fused_kernels.cuh -- the fused persistent sweep kernels: ONE CTA per space-time subdomain runs
// the whole window (forward: all W steps; adjoint: all W steps backwards) in one launch.
//
// Design ("row marching"): thread i of the CTA owns padded column i of
// the tile and marches over the rows.  All sub-stages of a step run software-pipelined on
// different rows in the same tick, so one __syncthreads per row:
//   forward  tick t : load Z0[t] | stage A row t-1 | h1 row t-2 | u1,v1 row t-3 -> store
//   adjoint  tick t : load Z0[t] | stage A row t-1, UB row t-1 | HB,P row t-2 | A row t-3 |
//                     lam0 row t-4 -> store
// North/south neighbours are the thread's own rolling registers; east/west neighbours come from
// small shared-memory row rings written one tick earlier.  HBM sees each trajectory level once
// per sweep direction (write in the forward kernel, read in the adjoint kernel) plus the frozen
// ghost ring; the adjoint variable lives in the gradient array (L2-resident while its CTA runs)
// and is updated in place, row j being rewritten three ticks after it was read.
// No step is recomputed, nothing is re-read from HBM, no atomics: results are deterministic.
#pragma once
#include <stdlib.h>
#include <string.h>
#include "common.cuh"
#include "model_math.cuh"

#define FK_NT 128          // threads per CTA = maximum padded tile width
#define FK_ZR 8            // depth of the Z0 row ring (adjoint reads rows t-5 .. t)

struct FusedPlan {
    int enabled = 0;
    int maxpy = 0, maxncell = 0;
    int lam_smem = 0;                 // adjoint variable resident in shared memory
    size_t smem_fwd = 0, smem_adj = 0;
    // persistent CTAs: one L2-persistent scratch slot per resident CTA (in-place state / adjoint variable)
    int nslots = 0, nslots_fwd = 0;
    long long slot_stride = 0;        // doubles
    double* scratch = nullptr;
    int* counter = nullptr;
};
#define FK_SLOTS (148 * 3)          // B200: 148 SMs x 3 resident CTAs (adjoint)
#define FK_SLOTS_FWD (148 * 4)      // forward kernel: 4 resident CTAs per SM
typedef void* (*fused_take_fn)(void* arena, size_t bytes);

inline bool fused_fits(const Sub* subs, int nsub)
{
    for (int k = 0; k < nsub; ++k)
        if (subs[k].px > FK_NT || subs[k].py < 1) return false;
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

// row tables of the tile in shared memory: entry r = padded row r-1 (rows -1 .. py, clamped)
struct FkTab {
    const double *dtcz, *gdtcz, *dtf, *dtt, *rp, *rm;
};
__device__ __forceinline__ FkTab fk_tables(const ModelP& m, const FkGeo& g, double* sm)
{
    const int TP = g.py + 2;
    for (int r = threadIdx.x; r < TP; r += FK_NT) {
        int gj = g.joff + r - 1;
        gj = gj < 0 ? 0 : (gj >= m.nlat ? m.nlat - 1 : gj);
        sm[r] = m.dtcz[gj]; sm[TP + r] = m.gdtcz[gj]; sm[2 * TP + r] = m.dtf[gj];
        sm[3 * TP + r] = m.dtt[gj]; sm[4 * TP + r] = m.rp[gj]; sm[5 * TP + r] = m.rm[gj];
    }
    FkTab t;
    t.dtcz = sm + 1; t.gdtcz = sm + TP + 1; t.dtf = sm + 2 * TP + 1; t.dtt = sm + 3 * TP + 1;
    t.rp = sm + 4 * TP + 1; t.rm = sm + 5 * TP + 1;
    return t;
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

// ------------------------------------------------------------------------------------------
// forward sweep of one window: Z^{n+1} = Phi(Z^n) for n = 0..W-1, every level to the store
__global__ void __launch_bounds__(FK_NT) fk_forward(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                    ModelP m, const double* __restrict__ x, double* traj,
                                                    const double* ghost)
{
    extern __shared__ double dsm[];
    __shared__ double z0s[2][3][FK_NT];
    __shared__ double uas[2][FK_NT];
    __shared__ double h1s[2][FK_NT];
    const int k = blockIdx.x;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const FkGeo g = fk_geo(s);
    const FkTab tb = fk_tables(m, g, dsm);
    const int i = g.i;
    const double kap = m.kap, dtcm = m.dtcm, gdtcm = m.gdtcm;
    // level 0 of the store = the control
    for (int c = threadIdx.x; c < 3 * s.ncell; c += FK_NT) traj[s.toff + c] = x[s.coff + c];
    __syncthreads();
    for (int n = 0; n < s.W; ++n) {
        const double* tz = traj + s.toff + (long long)n * 3 * s.ncell;
        double* tn = traj + s.toff + (long long)(n + 1) * 3 * s.ncell + (g.cU ? g.li : 0);
        const FkCol col = fk_col(g, tz, ghost + s.goff + (long long)n * 3 * s.nring);
        double zm[3] = { 0, 0, 0 }, zc[3] = { 0, 0, 0 }, zp[3] = { 0, 0, 0 }, zn[3] = { 0, 0, 0 };
        double ha1 = 0, ha2 = 0, ua1 = 0, ua2 = 0, ua3 = 0, va1 = 0, va2 = 0, va3 = 0;
        double h1a = 0, h1b = 0, h1c = 0;
        fk_load_row(g, col, 0, zn);
        for (int t = 0; t < s.py + 3; ++t) {
            // ---- S0: row t arrives (prefetched last tick), next row is requested
#pragma unroll
            for (int f = 0; f < 3; ++f) { zm[f] = zc[f]; zc[f] = zp[f]; zp[f] = zn[f]; }
            if (t == s.py && g.wn) { zp[0] = zc[0]; zp[1] = zc[1]; zp[2] = -zc[2]; }   // mirrored pole row
            if (t + 1 < s.py) fk_load_row(g, col, t + 1, zn);
            if (t < s.py) {
#pragma unroll
                for (int f = 0; f < 3; ++f) z0s[t & 1][f][i] = zp[f];
            }
            // ---- S1: stage A on row j = t-1
            {
                const int j = t - 1;
                double ha = 0, ua = 0, va = 0;
                if (j >= g.jA0 && j < g.jA1) {
                    double sm0 = zm[0], sm1 = zm[1], sm2 = zm[2];
                    if (j == 0 && g.ws) { sm0 = zc[0]; sm1 = zc[1]; sm2 = -zc[2]; }
                    const double cu = tb.dtcz[j] * zc[1], cv = dtcm * zc[2];
                    const double* zE = &z0s[j & 1][0][g.iE];
                    const double* zW = &z0s[j & 1][0][g.iW];
                    ha = mm_stageA(zc[0], zE[0], zW[0], zp[0], sm0, cu, cv, kap);
                    ua = mm_stageA(zc[1], zE[FK_NT], zW[FK_NT], zp[1], sm1, cu, cv, kap);
                    va = mm_stageA(zc[2], zE[2 * FK_NT], zW[2 * FK_NT], zp[2], sm2, cu, cv, kap);
                    uas[j & 1][i] = ua;
                }
                ha2 = ha1; ha1 = ha; ua3 = ua2; ua2 = ua1; ua1 = ua; va3 = va2; va2 = va1; va1 = va;
            }
            // ---- S2: h1 on row j = t-2
            {
                const int j = t - 2;
                double h1 = 0;
                if (j >= g.jH0 && j < g.jH1) {
                    const double vaN = (j == s.py - 1 && g.wn) ? -va2 : va1;
                    const double vaS = (j == 0 && g.ws) ? -va2 : va3;
                    const double D = mm_div(uas[j & 1][g.iE], uas[j & 1][g.iW], vaN, vaS, tb.dtcz[j], dtcm,
                                            tb.rp[j], tb.rm[j]);
                    h1 = mm_h1(ha2, D);
                    h1s[j & 1][i] = h1;
                }
                h1c = h1b; h1b = h1a; h1a = h1;
            }
            // ---- S3: u1, v1 on row j = t-3 -> trajectory store
            {
                const int j = t - 3;
                if (j >= g.jU0 && j < g.jU1) {
                    const double dtf = tb.dtf[j], dtt = tb.dtt[j];
                    const double h1N = (j == s.py - 1 && g.wn) ? h1b : h1a;
                    const double h1S = (j == 0 && g.ws) ? h1b : h1c;
                    const double u1 = mm_u1(ua3, va3, h1s[j & 1][g.iE], h1s[j & 1][g.iW], tb.gdtcz[j], dtf, dtt);
                    const double v1 = mm_v1(va3, u1, h1N, h1S, gdtcm, dtf, dtt);
                    if (g.cU) {
                        double* o = tn + (j - s.gys) * s.ex;
                        o[0] = h1b; o[s.ncell] = u1; o[2 * s.ncell] = v1;
                    }
                }
            }
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------
// adjoint sweep of one window.  The adjoint variable on the extended tile, [3][ncell], is updated
// in place level by level; LSM = it lives in shared memory (tiles up to ~100 KB), otherwise in
// the gradient array of the subdomain (L2-resident while its CTA runs).
template <bool LSM>
__global__ void __launch_bounds__(FK_NT) fk_adjoint(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                    ModelP m, CostP cp, GeoP geo, const double* __restrict__ x,
                                                    const double* __restrict__ xbs,
                                                    const double* __restrict__ xfrozen,
                                                    const double* __restrict__ pred_end, const double* traj,
                                                    const double* ghost,
                                                    const long long* __restrict__ obs_start,
                                                    const int* __restrict__ obs_idx,
                                                    const double* __restrict__ obs_y,
                                                    const double* __restrict__ obs_c, double* gx, double* gw)
{
    extern __shared__ double dsm[];
    __shared__ double zr[FK_ZR][3][FK_NT];
    __shared__ double uas[4][FK_NT];
    __shared__ double ubs[2][FK_NT];
    __shared__ double ps[2][FK_NT];
    __shared__ double as[2][3][FK_NT];
    const int k = blockIdx.x;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const FkGeo g = fk_geo(s);
    const FkTab tb = fk_tables(m, g, dsm);
    const int i = g.i;
    const int n3 = 3 * s.ncell, nc1 = s.ncell;
    double* lam = LSM ? dsm + 6 * (s.py + 2) : gx + s.coff;
    const double kap = m.kap, dtcm = m.dtcm, gdtcm = m.gdtcm, c0 = 1.0 - 4.0 * m.kap;
    // ---- adjoint variable at the window end: successor-window overlap forcing (25c), else zero
    {
        const bool succ = s.jw < geo.q - 1;
        const double* tw = traj + s.toff + (long long)s.W * n3;
        const double* xn = succ ? xfrozen + subs[k + geo.p1 * geo.p2].coff : nullptr;
        for (int c = threadIdx.x; c < n3; c += FK_NT) {
            const int f = c / s.ncell;
            lam[c] = succ ? 2.0 * cp.mu * (tw[c] - xn[c]) * cp.ib[f] : 0.0;
        }
        __syncthreads();
    }
    double* lcol = lam + (g.cU ? g.li : 0);                 // this thread's column of lam
    for (int n = s.W; n >= 0; --n) {
        // ---- H^T R^-1 (misfit) at level n (25b)
        if (obs_start) {
            const long long q0 = obs_start[s.ooff + n], q1 = obs_start[s.ooff + n + 1];
            const double* t = traj + s.toff + (long long)n * n3;
            for (long long q = q0 + threadIdx.x; q < q1; q += FK_NT) {
                const int idx = obs_idx[q];
                lam[idx] += 2.0 * obs_c[q] * (t[idx] - obs_y[q]);
            }
            __syncthreads();
        }
        if (n == 0) break;
        // ---- lam <- M_{n-1}^T lam, marching over the rows
        const double* tz = traj + s.toff + (long long)(n - 1) * n3;
        const double* tu = traj + s.toff + (long long)n * n3 + s.ncell + (g.cU ? g.li : 0);   // u^1
        const FkCol col = fk_col(g, tz, ghost + s.goff + (long long)(n - 1) * 3 * s.nring);
        double zm[3] = { 0, 0, 0 }, zc[3] = { 0, 0, 0 }, zp[3] = { 0, 0, 0 }, zn[3] = { 0, 0, 0 };
        double ha1 = 0, ha2 = 0, ua1 = 0, ua2 = 0, ua3 = 0, va1 = 0, va2 = 0, va3 = 0, va4 = 0;
        double hb1 = 0, hb2 = 0, vb1 = 0, vb2 = 0, vb3 = 0, UB1 = 0, UB2 = 0, UB3 = 0;
        double HB2 = 0, HB3 = 0, P2 = 0, P3 = 0, P4 = 0;
        double A3[3] = { 0, 0, 0 }, A4[3] = { 0, 0, 0 }, A5[3] = { 0, 0, 0 };
        double l0 = 0, l1 = 0, l2 = 0, l3 = 0;     // prefetched lam row (h,u,v) and u1
        fk_load_row(g, col, 0, zn);
        if (g.jU0 == 0) { l0 = lcol[0]; l1 = lcol[nc1]; l2 = lcol[2 * nc1]; l3 = tu[0]; }
        for (int t = 0; t < s.py + 4; ++t) {
            // ---- S0: row t of Z0
#pragma unroll
            for (int f = 0; f < 3; ++f) { zm[f] = zc[f]; zc[f] = zp[f]; zp[f] = zn[f]; }
            if (t == s.py && g.wn) { zp[0] = zc[0]; zp[1] = zc[1]; zp[2] = -zc[2]; }
            if (t + 1 < s.py) fk_load_row(g, col, t + 1, zn);
            if (t < s.py) {
#pragma unroll
                for (int f = 0; f < 3; ++f) zr[t & (FK_ZR - 1)][f][i] = zp[f];
            }
            // ---- S1: stage A and UB on row j = t-1
            {
                const int j = t - 1;
                double ha = 0, ua = 0, va = 0;
                if (j >= g.jA0 && j < g.jA1) {
                    double sm0 = zm[0], sm1 = zm[1], sm2 = zm[2];
                    if (j == 0 && g.ws) { sm0 = zc[0]; sm1 = zc[1]; sm2 = -zc[2]; }
                    const double cu = tb.dtcz[j] * zc[1], cv = dtcm * zc[2];
                    const double* zE = &zr[j & (FK_ZR - 1)][0][g.iE];
                    const double* zW = &zr[j & (FK_ZR - 1)][0][g.iW];
                    ha = mm_stageA(zc[0], zE[0], zW[0], zp[0], sm0, cu, cv, kap);
                    ua = mm_stageA(zc[1], zE[FK_NT], zW[FK_NT], zp[1], sm1, cu, cv, kap);
                    va = mm_stageA(zc[2], zE[2 * FK_NT], zW[2 * FK_NT], zp[2], sm2, cu, cv, kap);
                    uas[j & 3][i] = ua;
                }
                ha2 = ha1; ha1 = ha; ua3 = ua2; ua2 = ua1; ua1 = ua;
                va4 = va3; va3 = va2; va2 = va1; va1 = va;
                // lam row j (prefetched) -> UB; next row requested
                double UB = 0, hb = 0, vb = 0;
                if (j >= g.jU0 && j < g.jU1) {
                    if (g.cU) { hb = l0; vb = l2; UB = mm_UB(l1, l2, l3, tb.dtf[j], tb.dtt[j]); }
                }
                if (j + 1 >= g.jU0 && j + 1 < g.jU1) {
                    const int o = (j + 1 - s.gys) * s.ex;
                    l0 = lcol[o]; l1 = lcol[nc1 + o]; l2 = lcol[2 * nc1 + o]; l3 = tu[o];
                }
                hb2 = hb1; hb1 = hb; vb3 = vb2; vb2 = vb1; vb1 = vb; UB3 = UB2; UB2 = UB1; UB1 = UB;
                if (j >= 0) ubs[j & 1][i] = UB;
            }
            // ---- S2: HB, P on row j = t-2 (range 1)
            {
                const int j = t - 2;
                double HB = 0, P = 0;
                if (j >= g.jA0 && j < g.jA1) {
                    const double vbN = (j == s.py - 1 && g.wn) ? -vb2 : vb1;
                    const double vbS = (j == 0 && g.ws) ? -vb2 : vb3;
                    HB = mm_HB(hb2, vbN, vbS, ubs[j & 1][g.iE], ubs[j & 1][g.iW], gdtcm, tb.gdtcz[j]);
                    P = -ha2 * HB;
                }
                HB3 = HB2; HB2 = HB; P4 = P3; P3 = P2; P2 = P;
                if (j >= 0) ps[j & 1][i] = P;
            }
            // ---- S3: A on row j = t-3 (range 1; A_h on range 2)
            {
                const int j = t - 3;
                double a0 = 0, a1 = 0, a2 = 0;
                if (j >= g.jA0 && j < g.jA1) {
                    const double dtcz = tb.dtcz[j], dtf = tb.dtf[j], dtt = tb.dtt[j];
                    const bool atN = (j == s.py - 1 && g.wn), atS = (j == 0 && g.ws);
                    if (j >= g.jH0 && j < g.jH1) {
                        const double vaN = atN ? -va3 : va2;
                        const double vaS = atS ? -va3 : va4;
                        const double D = mm_div(uas[j & 3][g.iE], uas[j & 3][g.iW], vaN, vaS, dtcz, dtcm,
                                                tb.rp[j], tb.rm[j]);
                        a0 = mm_Ah(HB3, D);
                    }
                    const double PSr = atS ? tb.rm[j] * P3 : tb.rp[j - 1] * P4;
                    const double PNr = atN ? tb.rp[j] * P3 : tb.rm[j + 1] * P2;
                    a1 = mm_Au(UB3, va3, ps[j & 1][g.iW], ps[j & 1][g.iE], dtt, dtcz);
                    a2 = mm_Av(vb3, UB3, ua3, PSr, PNr, dtf, dtt, dtcm);
                }
#pragma unroll
                for (int f = 0; f < 3; ++f) { A5[f] = A4[f]; A4[f] = A3[f]; }
                A3[0] = a0; A3[1] = a1; A3[2] = a2;
                if (j >= 0) { as[j & 1][0][i] = a0; as[j & 1][1][i] = a1; as[j & 1][2][i] = a2; }
            }
            // ---- S4: lam0 on row j = t-4 (extended tile) -> in place
            {
                const int j = t - 4;
                if (j >= g.jU0 && j < g.jU1) {
                    const double dtcz = tb.dtcz[j];
                    const bool atN = (j == s.py - 1 && g.wn), atS = (j == 0 && g.ws);
                    const double* zc_ = &zr[j & (FK_ZR - 1)][0][0];
                    const double* zN_ = atN ? zc_ : &zr[(j + 1) & (FK_ZR - 1)][0][0];
                    const double* zS_ = atS ? zc_ : &zr[(j - 1) & (FK_ZR - 1)][0][0];
                    double xE[3], xW[3], xN[3], xS[3];
#pragma unroll
                    for (int f = 0; f < 3; ++f) {
                        xE[f] = zc_[f * FK_NT + g.iE]; xW[f] = zc_[f * FK_NT + g.iW];
                        xN[f] = zN_[f * FK_NT + i]; xS[f] = zS_[f * FK_NT + i];
                    }
                    if (atN) xN[2] = -xN[2];
                    if (atS) xS[2] = -xS[2];
                    const double kW = kap - dtcz * xW[1], kE = kap + dtcz * xE[1];
                    const double kS = kap - dtcm * xS[2], kN = kap + dtcm * xN[2];
                    const double* aE = &as[j & 1][0][g.iE];
                    const double* aW = &as[j & 1][0][g.iW];
                    double out[3], su = 0.0, sv = 0.0;
#pragma unroll
                    for (int f = 0; f < 3; ++f) {
                        const double sg = f == 2 ? -1.0 : 1.0;
                        const double aN = atN ? sg * A4[f] : A3[f];
                        const double aS = atS ? sg * A4[f] : A5[f];
                        out[f] = A4[f] * c0 + aW[f * FK_NT] * kW + aE[f * FK_NT] * kE + aS * kS + aN * kN;
                        su += (xE[f] - xW[f]) * A4[f];
                        sv += (xN[f] - xS[f]) * A4[f];
                    }
                    if (g.cU) {
                        double* o = lcol + (j - s.gys) * s.ex;
                        o[0] = out[0]; o[nc1] = out[1] - dtcz * su; o[2 * nc1] = out[2] - dtcm * sv;
                    }
                }
            }
            __syncthreads();
        }
    }
    // ---- gradient at the window start: adjoint variable + (25a) + control-level (25c) terms
    {
        const bool pred = s.jw > 0;
        for (int c = threadIdx.x; c < s.ncell; c += FK_NT) {
            const int lj = c / s.ex, li = c - lj * s.ex;
            const int gi = imodd(s.ei0 + li, geo.nlon), gj = s.ej0 + lj;
            const int nc = geo.ncolcov[gi], nr = geo.nrowcov[gj];
            const double wsp = 1.0 / (double)(nc * nr);
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const long long o = s.coff + (long long)f * s.ncell + c;
                const double xv = x[o];
                double gg = lam[f * s.ncell + c];
                gg += 2.0 * wsp * (xv - xbs[o]) * cp.ib[f];
                if (nc * nr > 1)
                    for (int cb = 0; cb < nr; ++cb)
                        for (int ca = 0; ca < nc; ++ca) {
                            const int a2 = geo.colcov[4 * gi + ca], b2 = geo.rowcov[4 * gj + cb];
                            if (a2 == s.a && b2 == s.b) continue;
                            const Sub& s2 = subs[(s.jw * geo.p2 + b2) * geo.p1 + a2];
                            const int li2 = imodd(gi - s2.ei0, geo.nlon), lj2 = gj - s2.ej0;
                            gg += 2.0 * cp.mu * (xv - xfrozen[s2.coff + (long long)f * s2.ncell + lj2 * s2.ex + li2]) * cp.ib[f];
                        }
                if (pred) gg += 2.0 * cp.mu * (xv - pred_end[o]) * cp.ib[f];
                gx[o] = gg;
                if (gw) gw[o] = cp.sb[f] * gg;
            }
        }
    }
}

// Row tables in constant memory for the static-slot kernels: entry [k][gj + 1], with guard entries
// r+_{-1} = 1 and r-_{nlat} = 1 for the virtual mirrored pole rows.  Uniform (per-CTA) index ->
// constant-cache loads, which keep the tables off the L1TEX/shared-memory pipe.
#define FK_CTAB 1026
__constant__ double c_tab[6][FK_CTAB];
#define CT_DTCZ 0
#define CT_GDTCZ 1
#define CT_DTF 2
#define CT_DTT 3
#define CT_RP 4
#define CT_RM 5
__device__ __forceinline__ double ctab(int k, int cj, int j) { return c_tab[k][cj + j]; }

#include "fused_adjoint.cuh"
#include "fused_forward.cuh"

// dynamic shared memory of the two kernels (row tables, and the adjoint variable when resident)
inline size_t fused_smem_forward(int maxpy) { return sizeof(double) * 6 * (size_t)(maxpy + 2); }
inline size_t fused_smem_adjoint(int maxpy, int maxncell, bool lsm)
{
    return sizeof(double) * (6 * (size_t)(maxpy + 2) + (lsm ? 3 * (size_t)maxncell : 0));
}

// lam_mode: 0 auto (shared memory when two CTAs per SM still fit), 1 global, 2 shared
inline void fused_plan_init(FusedPlan& fp, const Sub* subs, int nsub, int lam_mode)
{
    fp = FusedPlan();
    if (!subs || nsub <= 0) return;
    fp.enabled = 1;
    for (int k = 0; k < nsub; ++k) {
        fp.maxpy = subs[k].py > fp.maxpy ? subs[k].py : fp.maxpy;
        fp.maxncell = subs[k].ncell > fp.maxncell ? subs[k].ncell : fp.maxncell;
    }
    const size_t stat = sizeof(double) * FK_NT * (FK_ZR * 3 + 4 + 2 + 2 + 6);
    const size_t with = fused_smem_adjoint(fp.maxpy, fp.maxncell, true) + stat;
    const bool can = with <= 227 * 1024;
    const bool two = with <= 113 * 1024;
    fp.lam_smem = lam_mode == 2 ? (can ? 1 : 0) : (lam_mode == 1 ? 0 : (two ? 1 : 0));
    fp.nslots = nsub < FK_SLOTS ? nsub : FK_SLOTS;
    fp.nslots_fwd = nsub < FK_SLOTS_FWD ? nsub : FK_SLOTS_FWD;
    fp.slot_stride = (3LL * fp.maxncell + 31) & ~31LL;
    fp.smem_fwd = fused_smem_forward(fp.maxpy);
    fp.smem_adj = fused_smem_adjoint(fp.maxpy, fp.maxncell, fp.lam_smem != 0);
}
// copy the row tables (host, 6 x nlat, order dtcz gdtcz dtf dtt rp rm) into constant memory
inline int fused_upload_tables(cudaStream_t stream, const double* h_tab, int nlat)
{
    if (nlat + 2 > FK_CTAB) return -1;
    static double buf[6][FK_CTAB];
    for (int k = 0; k < 6; ++k) {
        for (int q = 0; q < FK_CTAB; ++q) buf[k][q] = 0.0;
        for (int j = 0; j < nlat; ++j) buf[k][j + 1] = h_tab[(size_t)k * nlat + j];
        buf[k][0] = buf[k][1]; buf[k][nlat + 1] = buf[k][nlat];
    }
    buf[CT_RP][0] = 1.0; buf[CT_RM][nlat + 1] = 1.0;
    cudaStreamSynchronize(stream);
    return cudaMemcpyToSymbol(c_tab, buf, sizeof(buf)) == cudaSuccess ? 0 : -1;
}
inline int fused_setup(cudaStream_t stream, FusedPlan& fp, const Sub*)
{
    if (!fp.enabled) return 0;
    {   // keep the per-CTA scratch resident in L2; everything else streams through the rest
        int dev = 0; cudaGetDevice(&dev);
        cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
        size_t bytes = sizeof(double) * (size_t)fp.nslots_fwd * fp.slot_stride;
        size_t lim = bytes < (size_t)prop.persistingL2CacheMaxSize ? bytes : (size_t)prop.persistingL2CacheMaxSize;
        if (lim > 0 && !getenv("DD4DVAR_NO_L2PIN")) {
            cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, lim);
            cudaStreamAttrValue av; memset(&av, 0, sizeof(av));
            av.accessPolicyWindow.base_ptr = fp.scratch;
            av.accessPolicyWindow.num_bytes = bytes < (size_t)prop.accessPolicyMaxWindowSize ? bytes : (size_t)prop.accessPolicyMaxWindowSize;
            av.accessPolicyWindow.hitRatio = lim >= bytes ? 1.0f : (float)lim / (float)bytes;
            av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
            av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
            cudaStreamSetAttribute(stream, cudaStreamAttributeAccessPolicyWindow, &av);
            cudaGetLastError();
        }
    }
    cudaError_t e = cudaFuncSetAttribute(fk_adjoint<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)fused_smem_adjoint(fp.maxpy, fp.maxncell, true) <= 200 * 1024
                                             ? (int)fused_smem_adjoint(fp.maxpy, fp.maxncell, true) : 200 * 1024);
    if (e != cudaSuccess) return -1;
    e = cudaFuncSetAttribute(fk_adjoint<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem_adjoint(fp.maxpy, fp.maxncell, false));
    if (e != cudaSuccess) return -1;
    e = cudaFuncSetAttribute(fk_adjoint2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem_adjoint(fp.maxpy, fp.maxncell, false));
    if (e != cudaSuccess) return -1;
    e = cudaFuncSetAttribute(fk_forward2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fp.smem_fwd);
    if (e != cudaSuccess) return -1;
    e = cudaFuncSetAttribute(fk_forward, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fp.smem_fwd);
    return e == cudaSuccess ? 0 : -1;
}
