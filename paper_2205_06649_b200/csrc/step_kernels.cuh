// step_kernels.cuh -- block-tiled ONE-LAUNCH-PER-STEP kernels of the generic path: a CTA computes a
// 32x16 tile of one step (forward) or of one adjoint step entirely in shared memory, recomputing
// the halo of the intermediate stages (overlapped tiling).  They serve any tile size (the
// undecomposed grid, the 1x1x1 .. 4x4x4 layouts of config 4) with one launch where the per-stage
// kernels of generic_kernels.cuh need four to six, and are checked against them and the oracle.
// Same ranges, same gather-form adjoint (model_math.cuh), same padded-array conventions.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
#include "generic_kernels.cuh"
#include "model_math.cuh"

#define SK_TX 32
#define SK_TY 16
#define SK_NT 256

// value of padded cell (i, j) of field f at local level n: trajectory store inside the extended
// tile, frozen ghost ring outside (same enumeration as gk_fill_pad)
__device__ __forceinline__ double sk_z0(const Sub& s, const Reg& r, const double* __restrict__ t,
                                        const double* __restrict__ g, int f, int i, int j)
{
    if (is_interior(r, i, j)) return t[(long long)f * s.ncell + (j - s.gys) * s.ex + (i - s.gx)];
    int rr;
    if (j < s.gys) rr = j * s.px + i;
    else if (j >= s.gys + s.ey) rr = s.gys * s.px + (j - s.gys - s.ey) * s.px + i;
    else rr = (s.gys + s.gyn) * s.px + (j - s.gys) * (2 * s.gx) + (i < s.gx ? i : i - s.ex);
    return g[(long long)f * s.nring + rr];
}

// Windows of padded cells held in shared memory: columns wrap when the region is periodic, rows are
// clipped to the region (a pole wall mirrors inside).
__device__ __forceinline__ int sk_wrap(const Reg& r, int i) { return r.perx ? imodd(i, r.px) : i; }
__device__ __forceinline__ bool sk_inside(const Reg& r, int i, int j)
{
    return (r.perx || (i >= 0 && i < r.px)) && j >= 0 && j < r.py;
}
// neighbour rows with the wall mirror (returns the row itself and sign -1 at a wall)
__device__ __forceinline__ void sk_ns(const Reg& r, int j, int& jN, int& jS, double& sN, double& sS)
{
    jN = j + 1; jS = j - 1; sN = 1.0; sS = 1.0;
    if (r.wn && j == r.py - 1) { jN = j; sN = -1.0; }
    if (r.ws && j == 0) { jS = j; sS = -1.0; }
}
// range test in UNWRAPPED window coordinates (i may lie outside [0,px) when periodic)
__device__ __forceinline__ bool sk_range(const Reg& r, int k, int i, int j)
{
    if (j < 0 || j >= r.py) return false;
    if (r.perx) return in_range(r, k, 0, j);
    return i >= 0 && i < r.px && in_range(r, k, i, j);
}

// ------------------------------------------------------------------------------------------
// forward step n: Z^{n+1} = Phi(Z^n) on one 32x16 output tile (tx, ty) of subdomain s; shared memory: z0 [3][H0*W0],
// za [3][H1*W1], h1 [H2*W2] (a caller that loops over tiles needs no barrier between two calls: the first
// phase of a call writes z0 only, which the last phase of the previous call does not read)
#define SK_FWD_SMEM_DOUBLES (3 * (SK_TY + 6) * (SK_TX + 6) + 3 * (SK_TY + 4) * (SK_TX + 4) + (SK_TY + 2) * (SK_TX + 2))
__device__ __forceinline__ void sk_forward_tile(const Sub& s, int tx, int ty, int n, const ModelP& m, double* traj,
                                                const double* __restrict__ ghost, double* __restrict__ z0,
                                                double* __restrict__ za, double* __restrict__ h1)
{
    constexpr int W0 = SK_TX + 6, H0 = SK_TY + 6, W1 = SK_TX + 4, H1 = SK_TY + 4, W2 = SK_TX + 2, H2 = SK_TY + 2;
    constexpr int N0 = H0 * W0, N1 = H1 * W1;
    const Reg r = make_reg(s);
    const int oi = s.gx + tx * SK_TX, oj = s.gys + ty * SK_TY;      // first output cell (padded coords)
    if (oi >= s.gx + s.ex || oj >= s.gys + s.ey) return;
    const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
    const double* g = ghost + s.goff + (long long)n * DD_NF * s.nring;
    // ---- Z0 on the tile + 3
    for (int c = threadIdx.x; c < N0; c += SK_NT) {
        const int lj = c / W0, li = c - lj * W0;
        const int i = oi - 3 + li, j = oj - 3 + lj;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        if (sk_inside(r, i, j)) {
            const int iw = sk_wrap(r, i);
            v0 = sk_z0(s, r, t, g, 0, iw, j); v1 = sk_z0(s, r, t, g, 1, iw, j); v2 = sk_z0(s, r, t, g, 2, iw, j);
        }
        z0[c] = v0; z0[N0 + c] = v1; z0[2 * N0 + c] = v2;
    }
    __syncthreads();
    // ---- stage A on the tile + 2 (range 1)
    for (int c = threadIdx.x; c < N1; c += SK_NT) {
        const int lj = c / W1, li = c - lj * W1;
        const int i = oi - 2 + li, j = oj - 2 + lj;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        if (sk_range(r, 1, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int cc = (lj + 1) * W0 + li + 1, cN = (jN - oj + 3) * W0 + li + 1, cS = (jS - oj + 3) * W0 + li + 1;
            const double* zh = z0; const double* zu = z0 + N0; const double* zv = z0 + 2 * N0;
            const double cu = m.dtcz[r.joff + j] * zu[cc], cv = m.dtcm * zv[cc];
            a0 = mm_stageA(zh[cc], zh[cc + 1], zh[cc - 1], zh[cN], zh[cS], cu, cv, m.kap);
            a1 = mm_stageA(zu[cc], zu[cc + 1], zu[cc - 1], zu[cN], zu[cS], cu, cv, m.kap);
            a2 = mm_stageA(zv[cc], zv[cc + 1], zv[cc - 1], sN * zv[cN], sS * zv[cS], cu, cv, m.kap);
        }
        za[c] = a0; za[N1 + c] = a1; za[2 * N1 + c] = a2;
    }
    __syncthreads();
    // ---- h1 on the tile + 1 (range 2)
    for (int c = threadIdx.x; c < H2 * W2; c += SK_NT) {
        const int lj = c / W2, li = c - lj * W2;
        const int i = oi - 1 + li, j = oj - 1 + lj;
        double v = 0.0;
        if (sk_range(r, 2, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int cc = (lj + 1) * W1 + li + 1, cN = (jN - oj + 2) * W1 + li + 1, cS = (jS - oj + 2) * W1 + li + 1;
            const int gj = r.joff + j;
            const double* ua = za + N1; const double* va = za + 2 * N1;
            const double D = mm_div(ua[cc + 1], ua[cc - 1], sN * va[cN], sS * va[cS], m.dtcz[gj], m.dtcm,
                                    m.rp[gj], m.rm[gj]);
            v = mm_h1(za[cc], D);
        }
        h1[c] = v;
    }
    __syncthreads();
    // ---- u1, v1 on the tile (range 3 = extended tile) -> trajectory store
    double* tn = traj + s.toff + (long long)(n + 1) * DD_NF * s.ncell;
    for (int c = threadIdx.x; c < SK_TY * SK_TX; c += SK_NT) {
        const int lj = c / SK_TX, li = c - lj * SK_TX;
        const int i = oi + li, j = oj + lj;
        if (i >= s.gx + s.ex || j >= s.gys + s.ey) continue;
        int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
        const int ca = (lj + 2) * W1 + li + 2;
        const int ch = (lj + 1) * W2 + li + 1, chN = (jN - oj + 1) * W2 + li + 1, chS = (jS - oj + 1) * W2 + li + 1;
        const int gj = r.joff + j;
        const double dtf = m.dtf[gj], dtt = m.dtt[gj];
        const double u1 = mm_u1(za[N1 + ca], za[2 * N1 + ca], h1[ch + 1], h1[ch - 1], m.gdtcz[gj], dtf, dtt);
        const double v1 = mm_v1(za[2 * N1 + ca], u1, h1[chN], h1[chS], m.gdtcm, dtf, dtt);
        const int lc = (j - s.gys) * s.ex + (i - s.gx);
        tn[lc] = h1[ch]; tn[s.ncell + lc] = u1; tn[2LL * s.ncell + lc] = v1;
    }
}
__global__ void __launch_bounds__(SK_NT) sk_forward_step(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                         int n, ModelP m, double* traj, const double* __restrict__ ghost,
                                                         int tiles_x)
{
    __shared__ double smf[SK_FWD_SMEM_DOUBLES];
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    if (n >= s.W) return;
    sk_forward_tile(s, blockIdx.x % tiles_x, blockIdx.x / tiles_x, n, m, traj, ghost, smf,
                    smf + 3 * (SK_TY + 6) * (SK_TX + 6), smf + 3 * (SK_TY + 6) * (SK_TX + 6) + 3 * (SK_TY + 4) * (SK_TX + 4));
}
// The steps n0 .. n1-1 of every subdomain in ONE cooperative launch: persistent CTAs loop over the (subdomain, tile)
// pairs of a step, a grid-wide barrier separates the steps (the undecomposed forecast of 256 steps is otherwise 256
// launches of a 10-microsecond kernel).  Launched with cudaLaunchCooperativeKernel, grid <= resident CTAs.
__global__ void __launch_bounds__(SK_NT) sk_forward_multi(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                          int n0, int n1, ModelP m, double* traj,
                                                          const double* __restrict__ ghost, int tiles_x, int ntiles, int nsub)
{
    __shared__ double smf[SK_FWD_SMEM_DOUBLES];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    for (int n = n0; n < n1; ++n) {
        for (int q = blockIdx.x; q < ntiles * nsub; q += gridDim.x) {
            const int k = q / ntiles, tile = q - k * ntiles;
            if (mask && !mask[k]) continue;
            const Sub s = subs[k];
            if (n >= s.W) continue;
            sk_forward_tile(s, tile % tiles_x, tile / tiles_x, n, m, traj, ghost, smf,
                            smf + 3 * (SK_TY + 6) * (SK_TX + 6), smf + 3 * (SK_TY + 6) * (SK_TX + 6) + 3 * (SK_TY + 4) * (SK_TX + 4));
        }
        grid.sync();
    }
}

// ------------------------------------------------------------------------------------------
// adjoint of step n (levels n+1 -> n) on one 32x16 output tile.  lam1 / lam0: padded [3][npad]
// arrays (zero on the ghost ring), as in gk_adjHB / gk_adjA / gk_adjL0.
#define SK_ADJ_SMEM_DOUBLES (3 * (SK_TY + 8) * (SK_TX + 8) + 6 * (SK_TY + 6) * (SK_TX + 6) + 2 * (SK_TY + 4) * (SK_TX + 4) + \
                             3 * (SK_TY + 2) * (SK_TX + 2))
__global__ void __launch_bounds__(SK_NT) sk_adjoint_step(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                         int n, ModelP m, const double* __restrict__ traj,
                                                         const double* __restrict__ ghost,
                                                         const double* __restrict__ lam1, double* __restrict__ lam0,
                                                         int tiles_x)
{
    constexpr int W0 = SK_TX + 8, H0 = SK_TY + 8, W1 = SK_TX + 6, H1 = SK_TY + 6, W2 = SK_TX + 4, H2 = SK_TY + 4,
                  W3 = SK_TX + 2, H3 = SK_TY + 2;
    extern __shared__ double sk_sm[];
    double* z0 = sk_sm;                       // [3][H0*W0]   tile + 4
    double* za = z0 + 3 * H0 * W0;            // [3][H1*W1]   tile + 3
    double* l1 = za + 3 * H1 * W1;            // [3][H1*W1]   hb1, UB, vb on tile + 3
    double* hb = l1 + 3 * H1 * W1;            // [H2*W2]      tile + 2
    double* pp = hb + H2 * W2;                // [H2*W2]
    double* aa = pp + H2 * W2;                // [3][H3*W3]   tile + 1
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    if (n >= s.W) return;
    const Reg r = make_reg(s);
    const int tx = blockIdx.x % tiles_x, ty = blockIdx.x / tiles_x;
    const int oi = s.gx + tx * SK_TX, oj = s.gys + ty * SK_TY;
    if (oi >= s.gx + s.ex || oj >= s.gys + s.ey) return;
    const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
    const double* g = ghost + s.goff + (long long)n * DD_NF * s.nring;
    const double* u1 = traj + s.toff + (long long)(n + 1) * DD_NF * s.ncell + s.ncell;
    const double* l1g = lam1 + s.poff;
    const long long np = s.npad;
    for (int c = threadIdx.x; c < H0 * W0; c += SK_NT) {
        const int lj = c / W0, li = c - lj * W0;
        const int i = oi - 4 + li, j = oj - 4 + lj;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        if (sk_inside(r, i, j)) {
            const int iw = sk_wrap(r, i);
            v0 = sk_z0(s, r, t, g, 0, iw, j); v1 = sk_z0(s, r, t, g, 1, iw, j); v2 = sk_z0(s, r, t, g, 2, iw, j);
        }
        z0[c] = v0; z0[H0 * W0 + c] = v1; z0[2 * H0 * W0 + c] = v2;
    }
    for (int c = threadIdx.x; c < H1 * W1; c += SK_NT) {
        const int lj = c / W1, li = c - lj * W1;
        const int i = oi - 3 + li, j = oj - 3 + lj;
        double h = 0.0, ub = 0.0, vb = 0.0;
        if (sk_inside(r, i, j)) {
            const int iw = sk_wrap(r, i);
            if (is_interior(r, iw, j)) {
                const int pc = j * s.px + iw, gj = r.joff + j;
                h = l1g[pc]; vb = l1g[2 * np + pc];
                ub = mm_UB(l1g[np + pc], vb, u1[(j - s.gys) * s.ex + (iw - s.gx)], m.dtf[gj], m.dtt[gj]);
            }
        }
        l1[c] = h; l1[H1 * W1 + c] = ub; l1[2 * H1 * W1 + c] = vb;
    }
    __syncthreads();
    // ---- stage A on tile + 3 (range 1)
    for (int c = threadIdx.x; c < H1 * W1; c += SK_NT) {
        const int lj = c / W1, li = c - lj * W1;
        const int i = oi - 3 + li, j = oj - 3 + lj;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        if (sk_range(r, 1, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int cc = (lj + 1) * W0 + li + 1, cN = (jN - oj + 4) * W0 + li + 1, cS = (jS - oj + 4) * W0 + li + 1;
            const double* zh = z0; const double* zu = z0 + H0 * W0; const double* zv = z0 + 2 * H0 * W0;
            const double cu = m.dtcz[r.joff + j] * zu[cc], cv = m.dtcm * zv[cc];
            a0 = mm_stageA(zh[cc], zh[cc + 1], zh[cc - 1], zh[cN], zh[cS], cu, cv, m.kap);
            a1 = mm_stageA(zu[cc], zu[cc + 1], zu[cc - 1], zu[cN], zu[cS], cu, cv, m.kap);
            a2 = mm_stageA(zv[cc], zv[cc + 1], zv[cc - 1], sN * zv[cN], sS * zv[cS], cu, cv, m.kap);
        }
        za[c] = a0; za[H1 * W1 + c] = a1; za[2 * H1 * W1 + c] = a2;
    }
    __syncthreads();
    // ---- HB, P on tile + 2 (range 1)
    for (int c = threadIdx.x; c < H2 * W2; c += SK_NT) {
        const int lj = c / W2, li = c - lj * W2;
        const int i = oi - 2 + li, j = oj - 2 + lj;
        double H = 0.0, P = 0.0;
        if (sk_range(r, 1, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int cc = (lj + 1) * W1 + li + 1, cN = (jN - oj + 3) * W1 + li + 1, cS = (jS - oj + 3) * W1 + li + 1;
            const double* vb = l1 + 2 * H1 * W1; const double* ub = l1 + H1 * W1;
            H = mm_HB(l1[cc], sN * vb[cN], sS * vb[cS], ub[cc + 1], ub[cc - 1], m.gdtcm, m.gdtcz[r.joff + j]);
            P = -za[cc] * H;
        }
        hb[c] = H; pp[c] = P;
    }
    __syncthreads();
    // ---- A on tile + 1 (range 1; A_h on range 2)
    for (int c = threadIdx.x; c < H3 * W3; c += SK_NT) {
        const int lj = c / W3, li = c - lj * W3;
        const int i = oi - 1 + li, j = oj - 1 + lj;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        if (sk_range(r, 1, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int gj = r.joff + j;
            const int ca = (lj + 2) * W1 + li + 2, caN = (jN - oj + 3) * W1 + li + 2, caS = (jS - oj + 3) * W1 + li + 2;
            const int cp_ = (lj + 1) * W2 + li + 1, cpN = (jN - oj + 2) * W2 + li + 1, cpS = (jS - oj + 2) * W2 + li + 1;
            const double* ua = za + H1 * W1; const double* va = za + 2 * H1 * W1;
            const double dtcz = m.dtcz[gj], dtf = m.dtf[gj], dtt = m.dtt[gj];
            if (sk_range(r, 2, i, j)) {
                const double D = mm_div(ua[ca + 1], ua[ca - 1], sN * va[caN], sS * va[caS], dtcz, m.dtcm, m.rp[gj], m.rm[gj]);
                a0 = mm_Ah(hb[cp_], D);
            }
            const double UBc = l1[H1 * W1 + ca], vbc = l1[2 * H1 * W1 + ca];
            const double PSr = (jS == j) ? m.rm[gj] * pp[cp_] : m.rp[gj - 1] * pp[cpS];
            const double PNr = (jN == j) ? m.rp[gj] * pp[cp_] : m.rm[gj + 1] * pp[cpN];
            a1 = mm_Au(UBc, va[ca], pp[cp_ - 1], pp[cp_ + 1], dtt, dtcz);
            a2 = mm_Av(vbc, UBc, ua[ca], PSr, PNr, dtf, dtt, m.dtcm);
        }
        aa[c] = a0; aa[H3 * W3 + c] = a1; aa[2 * H3 * W3 + c] = a2;
    }
    __syncthreads();
    // ---- lam0 on the tile (extended-tile cells only)
    double* l0 = lam0 + s.poff;
    for (int c = threadIdx.x; c < SK_TY * SK_TX; c += SK_NT) {
        const int lj = c / SK_TX, li = c - lj * SK_TX;
        const int i = oi + li, j = oj + lj;
        if (i >= s.gx + s.ex || j >= s.gys + s.ey) continue;
        int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
        const int cz = (lj + 4) * W0 + li + 4, czN = (jN - oj + 4) * W0 + li + 4, czS = (jS - oj + 4) * W0 + li + 4;
        const int ca = (lj + 1) * W3 + li + 1, caN = (jN - oj + 1) * W3 + li + 1, caS = (jS - oj + 1) * W3 + li + 1;
        const double dtcz = m.dtcz[r.joff + j], dtcm = m.dtcm;
        const double* zu = z0 + H0 * W0; const double* zv = z0 + 2 * H0 * W0;
        const double cuW = dtcz * zu[cz - 1], cuE = dtcz * zu[cz + 1];
        const double cvS = dtcm * sS * zv[czS], cvN = dtcm * sN * zv[czN];
        double out[3], su = 0.0, sv = 0.0;
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            const double* af = aa + f * H3 * W3; const double* zf = z0 + f * H0 * W0;
            const double mN = f == 2 ? sN : 1.0, mS = f == 2 ? sS : 1.0;
            out[f] = mm_L0(af[ca], af[ca - 1], af[ca + 1], mS * af[caS], mN * af[caN], cuW, cuE, cvS, cvN, m.kap);
            su += (zf[cz + 1] - zf[cz - 1]) * af[ca];
            sv += (mN * zf[czN] - mS * zf[czS]) * af[ca];
        }
        const int pc = j * s.px + i;
        l0[pc] = out[0]; l0[np + pc] = out[1] - dtcz * su; l0[2 * np + pc] = out[2] - dtcm * sv;
    }
}
