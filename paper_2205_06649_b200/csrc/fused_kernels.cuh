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
#include "common.cuh"
#include "model_math.cuh"

#define FK_NT 128          // threads per CTA = maximum padded tile width
#define FK_ZR 8            // depth of the Z0 row ring (adjoint reads rows t-5 .. t)

struct FusedPlan {
    int enabled = 0;
};
typedef void* (*fused_take_fn)(void* arena, size_t bytes);

inline bool fused_fits(const Sub* subs, int nsub)
{
    for (int k = 0; k < nsub; ++k)
        if (subs[k].px > FK_NT || subs[k].py < 1) return false;
    return nsub > 0;
}
inline void fused_plan_init(FusedPlan& fp, const Sub* subs, int nsub, int) { fp.enabled = subs && nsub > 0; }
inline void fused_plan_arrays(FusedPlan&, fused_take_fn, void*) {}

// geometry of the marching CTA, shared by both kernels
struct FkGeo {
    int px, py, ex, ey, gx, gys, gyn, joff, ncell, nring;
    bool perx, ws, wn;
    int i, li, iE, iW;
    bool col_ok, cA, cH, cU;
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
    g.cA = g.col_ok && (g.perx || (g.i >= 1 && g.i < s.px - 1));
    g.cH = g.col_ok && (g.perx || (g.i >= 2 && g.i < s.px - 2));
    g.cU = g.col_ok && g.li >= 0 && g.li < s.ex;
    return g;
}
__device__ __forceinline__ bool fk_vA(const FkGeo& g, int j) { return j >= (g.ws ? 0 : 1) && j < (g.wn ? g.py : g.py - 1); }
__device__ __forceinline__ bool fk_vH(const FkGeo& g, int j) { return j >= (g.ws ? 0 : 2) && j < (g.wn ? g.py : g.py - 2); }
__device__ __forceinline__ bool fk_vU(const FkGeo& g, int j) { return j >= g.gys && j < g.gys + g.ey; }

// value of padded row j, column of this thread, from the trajectory level (interior) or the frozen
// ghost ring of that level
__device__ __forceinline__ void fk_load_row(const FkGeo& g, int j, const double* tz, const double* gz, double z[3])
{
    z[0] = z[1] = z[2] = 0.0;
    if (!g.col_ok || j < 0 || j >= g.py) return;
    if (j >= g.gys && j < g.gys + g.ey) {
        if (g.cU) {
            const int c = (j - g.gys) * g.ex + g.li;
#pragma unroll
            for (int f = 0; f < 3; ++f) z[f] = tz[(long long)f * g.ncell + c];
        } else {
            const int rr = (g.gys + g.gyn) * g.px + (j - g.gys) * (2 * g.gx) + (g.i < g.gx ? g.i : g.i - g.ex);
#pragma unroll
            for (int f = 0; f < 3; ++f) z[f] = __ldg(gz + (long long)f * g.nring + rr);
        }
    } else {
        const int rr = j < g.gys ? j * g.px + g.i : g.gys * g.px + (j - g.gys - g.ey) * g.px + g.i;
#pragma unroll
        for (int f = 0; f < 3; ++f) z[f] = __ldg(gz + (long long)f * g.nring + rr);
    }
}

// ------------------------------------------------------------------------------------------
// forward sweep of one window: Z^{n+1} = Phi(Z^n) for n = 0..W-1, every level to the store
__global__ void __launch_bounds__(FK_NT) fk_forward(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                    ModelP m, const double* __restrict__ x, double* traj,
                                                    const double* __restrict__ ghost)
{
    __shared__ double z0s[2][3][FK_NT];
    __shared__ double uas[2][FK_NT];
    __shared__ double h1s[2][FK_NT];
    const int k = blockIdx.x;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const FkGeo g = fk_geo(s);
    const int i = g.i;
    // level 0 of the store = the control
    for (int c = threadIdx.x; c < 3 * s.ncell; c += FK_NT) traj[s.toff + c] = x[s.coff + c];
    __syncthreads();
    for (int n = 0; n < s.W; ++n) {
        const double* tz = traj + s.toff + (long long)n * 3 * s.ncell;
        double* tn = traj + s.toff + (long long)(n + 1) * 3 * s.ncell;
        const double* gz = ghost + s.goff + (long long)n * 3 * s.nring;
        double zm[3] = { 0, 0, 0 }, zc[3] = { 0, 0, 0 }, zp[3] = { 0, 0, 0 }, zn[3];
        double ha1 = 0, ha2 = 0, ua1 = 0, ua2 = 0, ua3 = 0, va1 = 0, va2 = 0, va3 = 0;
        double h1a = 0, h1b = 0, h1c = 0;
        fk_load_row(g, 0, tz, gz, zn);
        for (int t = 0; t < s.py + 3; ++t) {
            // ---- S0: row t arrives (prefetched last tick), next row is requested
#pragma unroll
            for (int f = 0; f < 3; ++f) { zm[f] = zc[f]; zc[f] = zp[f]; zp[f] = zn[f]; }
            if (t == s.py && g.wn) { zp[0] = zc[0]; zp[1] = zc[1]; zp[2] = -zc[2]; }   // mirrored pole row
            fk_load_row(g, t + 1, tz, gz, zn);
            if (t < s.py) {
#pragma unroll
                for (int f = 0; f < 3; ++f) z0s[t & 1][f][i] = zp[f];
            }
            // ---- S1: stage A on row j = t-1
            {
                const int j = t - 1;
                double ha = 0, ua = 0, va = 0;
                if (g.cA && fk_vA(g, j)) {
                    const int gj = g.joff + j;
                    double sm0 = zm[0], sm1 = zm[1], sm2 = zm[2];
                    if (j == 0 && g.ws) { sm0 = zc[0]; sm1 = zc[1]; sm2 = -zc[2]; }
                    const double cu = m.dtcz[gj] * zc[1], cv = m.dtcm * zc[2];
                    ha = mm_stageA(zc[0], z0s[j & 1][0][g.iE], z0s[j & 1][0][g.iW], zp[0], sm0, cu, cv, m.kap);
                    ua = mm_stageA(zc[1], z0s[j & 1][1][g.iE], z0s[j & 1][1][g.iW], zp[1], sm1, cu, cv, m.kap);
                    va = mm_stageA(zc[2], z0s[j & 1][2][g.iE], z0s[j & 1][2][g.iW], zp[2], sm2, cu, cv, m.kap);
                }
                ha2 = ha1; ha1 = ha; ua3 = ua2; ua2 = ua1; ua1 = ua; va3 = va2; va2 = va1; va1 = va;
                if (j >= 0) uas[j & 1][i] = ua;
            }
            // ---- S2: h1 on row j = t-2
            {
                const int j = t - 2;
                double h1 = 0;
                if (g.cH && fk_vH(g, j)) {
                    const int gj = g.joff + j;
                    const double vaN = (j == s.py - 1 && g.wn) ? -va2 : va1;
                    const double vaS = (j == 0 && g.ws) ? -va2 : va3;
                    const double D = mm_div(uas[j & 1][g.iE], uas[j & 1][g.iW], vaN, vaS, m.dtcz[gj], m.dtcm,
                                            m.rp[gj], m.rm[gj]);
                    h1 = mm_h1(ha2, D);
                }
                h1c = h1b; h1b = h1a; h1a = h1;
                if (j >= 0) h1s[j & 1][i] = h1;
            }
            // ---- S3: u1, v1 on row j = t-3 -> trajectory store
            {
                const int j = t - 3;
                if (g.cU && fk_vU(g, j)) {
                    const int gj = g.joff + j;
                    const double dtf = m.dtf[gj], dtt = m.dtt[gj];
                    const double h1N = (j == s.py - 1 && g.wn) ? h1b : h1a;
                    const double h1S = (j == 0 && g.ws) ? h1b : h1c;
                    const double u1 = mm_u1(ua3, va3, h1s[j & 1][g.iE], h1s[j & 1][g.iW], m.gdtcz[gj], dtf, dtt);
                    const double v1 = mm_v1(va3, u1, h1N, h1S, m.gdtcm, dtf, dtt);
                    const int c = (j - s.gys) * s.ex + g.li;
                    tn[c] = h1b;
                    tn[s.ncell + c] = u1;
                    tn[2 * s.ncell + c] = v1;
                }
            }
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------
// adjoint sweep of one window.  lam (= the gradient array of this subdomain, [3][ncell]) holds
// the adjoint variable on the extended tile and is updated in place level by level.
__global__ void __launch_bounds__(FK_NT) fk_adjoint(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                    ModelP m, CostP cp, GeoP geo, const double* __restrict__ x,
                                                    const double* __restrict__ xbs,
                                                    const double* __restrict__ xfrozen,
                                                    const double* __restrict__ pred_end, const double* traj,
                                                    const double* __restrict__ ghost,
                                                    const long long* __restrict__ obs_start,
                                                    const int* __restrict__ obs_idx,
                                                    const double* __restrict__ obs_y,
                                                    const double* __restrict__ obs_c, double* gx, double* gw)
{
    __shared__ double zr[FK_ZR][3][FK_NT];
    __shared__ double uas[4][FK_NT];
    __shared__ double ubs[2][FK_NT];
    __shared__ double ps[2][FK_NT];
    __shared__ double as[2][3][FK_NT];
    const int k = blockIdx.x;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const FkGeo g = fk_geo(s);
    const int i = g.i;
    double* lam = gx + s.coff;
    const int n3 = 3 * s.ncell;
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
        const double* tu = traj + s.toff + (long long)n * n3 + s.ncell;      // u^1 = u of level n
        const double* gz = ghost + s.goff + (long long)(n - 1) * 3 * s.nring;
        double zm[3] = { 0, 0, 0 }, zc[3] = { 0, 0, 0 }, zp[3] = { 0, 0, 0 }, zn[3];
        double ha1 = 0, ha2 = 0, ua1 = 0, ua2 = 0, ua3 = 0, va1 = 0, va2 = 0, va3 = 0, va4 = 0;
        double hb1 = 0, hb2 = 0, vb1 = 0, vb2 = 0, vb3 = 0, UB1 = 0, UB2 = 0, UB3 = 0;
        double HB2 = 0, HB3 = 0, P2 = 0, P3 = 0, P4 = 0;
        double A3[3] = { 0, 0, 0 }, A4[3] = { 0, 0, 0 }, A5[3] = { 0, 0, 0 };
        double ln[4] = { 0, 0, 0, 0 };     // prefetched lam row (h,u,v) and u1
        fk_load_row(g, 0, tz, gz, zn);
        if (g.cU && fk_vU(g, 0)) {
            const int c = (0 - s.gys) * s.ex + g.li;
            ln[0] = lam[c]; ln[1] = lam[s.ncell + c]; ln[2] = lam[2 * s.ncell + c]; ln[3] = tu[c];
        }
        for (int t = 0; t < s.py + 4; ++t) {
            // ---- S0: row t of Z0
#pragma unroll
            for (int f = 0; f < 3; ++f) { zm[f] = zc[f]; zc[f] = zp[f]; zp[f] = zn[f]; }
            if (t == s.py && g.wn) { zp[0] = zc[0]; zp[1] = zc[1]; zp[2] = -zc[2]; }
            fk_load_row(g, t + 1, tz, gz, zn);
            if (t < s.py) {
#pragma unroll
                for (int f = 0; f < 3; ++f) zr[t & (FK_ZR - 1)][f][i] = zp[f];
            }
            // ---- S1: stage A and UB on row j = t-1
            {
                const int j = t - 1;
                double ha = 0, ua = 0, va = 0;
                if (g.cA && fk_vA(g, j)) {
                    const int gj = g.joff + j, r = j & (FK_ZR - 1);
                    double sm0 = zm[0], sm1 = zm[1], sm2 = zm[2];
                    if (j == 0 && g.ws) { sm0 = zc[0]; sm1 = zc[1]; sm2 = -zc[2]; }
                    const double cu = m.dtcz[gj] * zc[1], cv = m.dtcm * zc[2];
                    ha = mm_stageA(zc[0], zr[r][0][g.iE], zr[r][0][g.iW], zp[0], sm0, cu, cv, m.kap);
                    ua = mm_stageA(zc[1], zr[r][1][g.iE], zr[r][1][g.iW], zp[1], sm1, cu, cv, m.kap);
                    va = mm_stageA(zc[2], zr[r][2][g.iE], zr[r][2][g.iW], zp[2], sm2, cu, cv, m.kap);
                }
                ha2 = ha1; ha1 = ha; ua3 = ua2; ua2 = ua1; ua1 = ua;
                va4 = va3; va3 = va2; va2 = va1; va1 = va;
                if (j >= 0) uas[j & 3][i] = ua;
                // lam^{n} row j (prefetched) -> UB; next row requested
                double UB = 0, hb = 0, vb = 0;
                if (g.cU && fk_vU(g, j)) {
                    const int gj = g.joff + j;
                    hb = ln[0]; vb = ln[2];
                    UB = mm_UB(ln[1], ln[2], ln[3], m.dtf[gj], m.dtt[gj]);
                }
                if (g.cU && fk_vU(g, j + 1)) {
                    const int c = (j + 1 - s.gys) * s.ex + g.li;
                    ln[0] = lam[c]; ln[1] = lam[s.ncell + c]; ln[2] = lam[2 * s.ncell + c]; ln[3] = tu[c];
                }
                hb2 = hb1; hb1 = hb; vb3 = vb2; vb2 = vb1; vb1 = vb; UB3 = UB2; UB2 = UB1; UB1 = UB;
                if (j >= 0) ubs[j & 1][i] = UB;
            }
            // ---- S2: HB, P on row j = t-2 (range 1)
            {
                const int j = t - 2;
                double HB = 0, P = 0;
                if (g.cA && fk_vA(g, j)) {
                    const int gj = g.joff + j;
                    const double vbN = (j == s.py - 1 && g.wn) ? -vb2 : vb1;
                    const double vbS = (j == 0 && g.ws) ? -vb2 : vb3;
                    HB = mm_HB(hb2, vbN, vbS, ubs[j & 1][g.iE], ubs[j & 1][g.iW], m.gdtcm, m.gdtcz[gj]);
                    P = -ha2 * HB;
                }
                HB3 = HB2; HB2 = HB; P4 = P3; P3 = P2; P2 = P;
                if (j >= 0) ps[j & 1][i] = P;
            }
            // ---- S3: A on row j = t-3 (range 1; A_h on range 2)
            {
                const int j = t - 3;
                double a0 = 0, a1 = 0, a2 = 0;
                if (g.cA && fk_vA(g, j)) {
                    const int gj = g.joff + j;
                    const double dtcz = m.dtcz[gj], dtf = m.dtf[gj], dtt = m.dtt[gj];
                    const bool atN = (j == s.py - 1 && g.wn), atS = (j == 0 && g.ws);
                    if (g.cH && fk_vH(g, j)) {
                        const double vaN = atN ? -va3 : va2;
                        const double vaS = atS ? -va3 : va4;
                        const double D = mm_div(uas[j & 3][g.iE], uas[j & 3][g.iW], vaN, vaS, dtcz, m.dtcm,
                                                m.rp[gj], m.rm[gj]);
                        a0 = mm_Ah(HB3, D);
                    }
                    const double PSr = atS ? m.rm[gj] * P3 : m.rp[gj - 1] * P4;
                    const double PNr = atN ? m.rp[gj] * P3 : m.rm[gj + 1] * P2;
                    a1 = mm_Au(UB3, va3, ps[j & 1][g.iW], ps[j & 1][g.iE], dtt, dtcz);
                    a2 = mm_Av(vb3, UB3, ua3, PSr, PNr, dtf, dtt, m.dtcm);
                }
#pragma unroll
                for (int f = 0; f < 3; ++f) { A5[f] = A4[f]; A4[f] = A3[f]; }
                A3[0] = a0; A3[1] = a1; A3[2] = a2;
                if (j >= 0) { as[j & 1][0][i] = a0; as[j & 1][1][i] = a1; as[j & 1][2][i] = a2; }
            }
            // ---- S4: lam0 on row j = t-4 (extended tile) -> in place
            {
                const int j = t - 4;
                if (g.cU && fk_vU(g, j)) {
                    const int gj = g.joff + j;
                    const double dtcz = m.dtcz[gj], dtcm = m.dtcm;
                    const bool atN = (j == s.py - 1 && g.wn), atS = (j == 0 && g.ws);
                    const int r = j & (FK_ZR - 1), rN = (j + 1) & (FK_ZR - 1), rS = (j - 1) & (FK_ZR - 1);
                    double xE[3], xW[3], xN[3], xS[3];
#pragma unroll
                    for (int f = 0; f < 3; ++f) {
                        xE[f] = zr[r][f][g.iE]; xW[f] = zr[r][f][g.iW];
                        xN[f] = atN ? zr[r][f][i] : zr[rN][f][i];
                        xS[f] = atS ? zr[r][f][i] : zr[rS][f][i];
                    }
                    if (atN) xN[2] = -xN[2];
                    if (atS) xS[2] = -xS[2];
                    const double cuW = dtcz * xW[1], cuE = dtcz * xE[1];
                    const double cvS = dtcm * xS[2], cvN = dtcm * xN[2];
                    double out[3], su = 0.0, sv = 0.0;
#pragma unroll
                    for (int f = 0; f < 3; ++f) {
                        const double sg = f == 2 ? -1.0 : 1.0;
                        const double aN = atN ? sg * A4[f] : A3[f];
                        const double aS = atS ? sg * A4[f] : A5[f];
                        out[f] = mm_L0(A4[f], as[j & 1][f][g.iW], as[j & 1][f][g.iE], aS, aN, cuW, cuE, cvS, cvN, m.kap);
                        su += (xE[f] - xW[f]) * A4[f];
                        sv += (xN[f] - xS[f]) * A4[f];
                    }
                    const int c = (j - s.gys) * s.ex + g.li;
                    lam[c] = out[0];
                    lam[s.ncell + c] = out[1] - dtcz * su;
                    lam[2 * s.ncell + c] = out[2] - dtcm * sv;
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
                double gg = gx[o];
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

inline int fused_setup(cudaStream_t, FusedPlan&, const Sub*) { return 0; }
