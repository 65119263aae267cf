// generic_kernels.cuh -- the per-step, global-memory path: one launch per sub-stage, batched over
// all subdomains (blockIdx.y = subdomain), one thread per padded cell.  It serves every layout
// (any tile size, ragged tiles, the undecomposed global grid) and is the in-library cross-check
// of the fused persistent kernels.  Stage ranges follow DESIGN.md "Ranges": a side that is open
// (carries a ghost ring) loses one cell per sub-stage, a closed side (periodic longitude, pole
// wall) loses none.
#pragma once
#include "common.cuh"
#include "model_math.cuh"

struct Reg {
    int px, py, joff, perx, ws, wn, gx, gys, ex, ey;
};
__device__ __forceinline__ Reg make_reg(const Sub& s)
{
    Reg r;
    r.px = s.px; r.py = s.py; r.joff = s.ej0 - s.gys;
    r.perx = s.gx == 0; r.ws = s.gys == 0; r.wn = s.gyn == 0;
    r.gx = s.gx; r.gys = s.gys; r.ex = s.ex; r.ey = s.ey;
    return r;
}
__device__ __forceinline__ bool in_range(const Reg& r, int k, int i, int j)
{
    const int ox = r.perx ? 0 : k;
    const int j0 = r.ws ? 0 : k, j1 = r.wn ? r.py : r.py - k;
    return i >= ox && i < r.px - ox && j >= j0 && j < j1;
}
__device__ __forceinline__ bool is_interior(const Reg& r, int i, int j)
{
    return i >= r.gx && i < r.gx + r.ex && j >= r.gys && j < r.gys + r.ey;
}
// neighbour indices inside the padded array; sN/sS = sign applied to v-like quantities when the
// neighbour is the reflected pole row (then jN/jS = j itself)
struct Nb { int iE, iW, jN, jS; double sN, sS; };
__device__ __forceinline__ Nb nbrs(const Reg& r, int i, int j)
{
    Nb n;
    n.iE = i + 1; n.iW = i - 1;
    if (r.perx) { if (n.iE == r.px) n.iE = 0; if (n.iW < 0) n.iW = r.px - 1; }
    n.jN = j + 1; n.jS = j - 1; n.sN = 1.0; n.sS = 1.0;
    if (r.wn && j == r.py - 1) { n.jN = j; n.sN = -1.0; }
    if (r.ws && j == 0) { n.jS = j; n.sS = -1.0; }
    return n;
}

#define GK_PROLOGUE                                                         \
    const int k = blockIdx.y;                                               \
    if (mask && !mask[k]) return;                                           \
    const Sub s = subs[k];                                                  \
    const int pc = blockIdx.x * blockDim.x + threadIdx.x;                   \
    if (pc >= s.npad) return;                                               \
    const Reg r = make_reg(s);                                              \
    const int j = pc / s.px, i = pc - j * s.px;

// level 0 of the trajectory store = the control (the state at the window start, l.275)
__global__ void gk_store_control(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                 const double* __restrict__ x, double* __restrict__ traj)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.ncell) return;
#pragma unroll
    for (int f = 0; f < DD_NF; ++f)
        traj[s.toff + (long long)f * s.ncell + c] = x[s.coff + (long long)f * s.ncell + c];
}

// Z0 padded = interior from the trajectory store at local level n, ghost ring from the frozen
// ghost store (R14).
__global__ void gk_fill_pad(const Sub* __restrict__ subs, const int* __restrict__ mask, int n,
                            const double* __restrict__ traj, const double* __restrict__ ghost,
                            double* __restrict__ Zp)
{
    GK_PROLOGUE
    if (n >= s.W) return;
    double* zp = Zp + s.poff;
    if (is_interior(r, i, j)) {
        const int lc = (j - s.gys) * s.ex + (i - s.gx);
        const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
#pragma unroll
        for (int f = 0; f < DD_NF; ++f) zp[(long long)f * s.npad + pc] = t[(long long)f * s.ncell + lc];
    } else {
        int rr;
        if (j < s.gys) rr = j * s.px + i;
        else if (j >= s.gys + s.ey) rr = s.gys * s.px + (j - s.gys - s.ey) * s.px + i;
        else rr = (s.gys + s.gyn) * s.px + (j - s.gys) * (2 * s.gx) + (i < s.gx ? i : i - s.ex);
        const double* g = ghost + s.goff + (long long)n * DD_NF * s.nring;
#pragma unroll
        for (int f = 0; f < DD_NF; ++f) zp[(long long)f * s.npad + pc] = g[(long long)f * s.nring + rr];
    }
}

__global__ void gk_stageA(const Sub* __restrict__ subs, const int* __restrict__ mask, int n,
                          ModelP m, const double* __restrict__ Zp, double* __restrict__ Za)
{
    GK_PROLOGUE
    if (n >= s.W || !in_range(r, 1, i, j)) return;
    const double* z = Zp + s.poff;
    double* za = Za + s.poff;
    const Nb nb = nbrs(r, i, j);
    const int gj = r.joff + j;
    const long long np = s.npad;
    const double cu = m.dtcz[gj] * z[np + pc], cv = m.dtcm * z[2 * np + pc];
#pragma unroll
    for (int f = 0; f < DD_NF; ++f) {
        const double* zf = z + f * np;
        const double mN = f == 2 ? nb.sN : 1.0, mS = f == 2 ? nb.sS : 1.0;
        za[f * np + pc] = mm_stageA(zf[pc], zf[j * s.px + nb.iE], zf[j * s.px + nb.iW],
                                    mN * zf[nb.jN * s.px + i], mS * zf[nb.jS * s.px + i], cu, cv, m.kap);
    }
}

__global__ void gk_stageH(const Sub* __restrict__ subs, const int* __restrict__ mask, int n,
                          ModelP m, const double* __restrict__ Za, double* __restrict__ H1)
{
    GK_PROLOGUE
    if (n >= s.W || !in_range(r, 2, i, j)) return;
    const double* za = Za + s.poff;
    const Nb nb = nbrs(r, i, j);
    const int gj = r.joff + j;
    const long long np = s.npad;
    const double D = mm_div(za[np + j * s.px + nb.iE], za[np + j * s.px + nb.iW],
                            nb.sN * za[2 * np + nb.jN * s.px + i], nb.sS * za[2 * np + nb.jS * s.px + i],
                            m.dtcz[gj], m.dtcm, m.rp[gj], m.rm[gj]);
    H1[s.poff / 3 + pc] = mm_h1(za[pc], D);
}

// u1, v1 on range 3 (= the extended tile); the new level goes to the trajectory store
__global__ void gk_stageUV(const Sub* __restrict__ subs, const int* __restrict__ mask, int n,
                           ModelP m, const double* __restrict__ Za, const double* __restrict__ H1,
                           double* __restrict__ traj)
{
    GK_PROLOGUE
    if (n >= s.W || !is_interior(r, i, j)) return;
    const double* za = Za + s.poff;
    const double* h1 = H1 + s.poff / 3;
    const Nb nb = nbrs(r, i, j);
    const int gj = r.joff + j;
    const long long np = s.npad;
    const double ua = za[np + pc], va = za[2 * np + pc];
    const double dtf = m.dtf[gj], dtt = m.dtt[gj];
    const double u1 = mm_u1(ua, va, h1[j * s.px + nb.iE], h1[j * s.px + nb.iW], m.gdtcz[gj], dtf, dtt);
    const double v1 = mm_v1(va, u1, h1[nb.jN * s.px + i], h1[nb.jS * s.px + i], m.gdtcm, dtf, dtt);
    const int lc = (j - s.gys) * s.ex + (i - s.gx);
    double* t = traj + s.toff + (long long)(n + 1) * DD_NF * s.ncell;
    t[lc] = h1[pc];
    t[s.ncell + lc] = u1;
    t[2LL * s.ncell + lc] = v1;
}

// ------------------------------------------------------------------------------------------
// adjoint of step n (levels n+1 -> n).  lam1: padded [3][npad], zero on the ghost ring.
// HB, P, UB on range 1 (zero elsewhere).
__global__ void gk_adjHB(const Sub* __restrict__ subs, const int* __restrict__ mask, int n, ModelP m,
                         const double* __restrict__ Za, const double* __restrict__ lam1,
                         const double* __restrict__ traj, double* __restrict__ HB,
                         double* __restrict__ P, double* __restrict__ UB)
{
    GK_PROLOGUE
    if (n >= s.W) return;
    const long long p1 = s.poff / 3;
    if (!in_range(r, 1, i, j)) { HB[p1 + pc] = 0.0; P[p1 + pc] = 0.0; UB[p1 + pc] = 0.0; return; }
    const double* za = Za + s.poff;
    const double* l1 = lam1 + s.poff;
    const double* u1 = traj + s.toff + (long long)(n + 1) * DD_NF * s.ncell + s.ncell;
    const Nb nb = nbrs(r, i, j);
    const int gj = r.joff + j;
    const long long np = s.npad;
    const double dtf = m.dtf[gj], dtt = m.dtt[gj];
    double ub[3];
    const int ii[3] = { i, nb.iE, nb.iW };
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const int i2 = ii[q];
        if (is_interior(r, i2, j)) {
            const int c2 = j * s.px + i2;
            ub[q] = mm_UB(l1[np + c2], l1[2 * np + c2], u1[(j - s.gys) * s.ex + (i2 - s.gx)], dtf, dtt);
        } else ub[q] = 0.0;
    }
    const double vbN = nb.sN * l1[2 * np + nb.jN * s.px + i], vbS = nb.sS * l1[2 * np + nb.jS * s.px + i];
    const double hb = mm_HB(l1[pc], vbN, vbS, ub[1], ub[2], m.gdtcm, m.gdtcz[gj]);
    HB[p1 + pc] = hb;
    P[p1 + pc] = -za[pc] * hb;
    UB[p1 + pc] = ub[0];
}

__global__ void gk_adjA(const Sub* __restrict__ subs, const int* __restrict__ mask, int n, ModelP m,
                        const double* __restrict__ Za, const double* __restrict__ lam1,
                        const double* __restrict__ HB, const double* __restrict__ P,
                        const double* __restrict__ UB, double* __restrict__ A)
{
    GK_PROLOGUE
    if (n >= s.W) return;
    double* a = A + s.poff;
    const long long np = s.npad;
    if (!in_range(r, 1, i, j)) { a[pc] = 0.0; a[np + pc] = 0.0; a[2 * np + pc] = 0.0; return; }
    const long long p1 = s.poff / 3;
    const double* za = Za + s.poff;
    const double* hbp = HB + p1;
    const double* pp = P + p1;
    const Nb nb = nbrs(r, i, j);
    const int gj = r.joff + j;
    const double dtcz = m.dtcz[gj], dtf = m.dtf[gj], dtt = m.dtt[gj];
    const double ub = UB[p1 + pc];
    double a0 = 0.0;
    if (in_range(r, 2, i, j)) {
        const double D = mm_div(za[np + j * s.px + nb.iE], za[np + j * s.px + nb.iW],
                                nb.sN * za[2 * np + nb.jN * s.px + i], nb.sS * za[2 * np + nb.jS * s.px + i],
                                dtcz, m.dtcm, m.rp[gj], m.rm[gj]);
        a0 = mm_Ah(hbp[pc], D);
    }
    const double PSr = (nb.jS == j) ? m.rm[gj] * pp[pc] : m.rp[gj - 1] * pp[nb.jS * s.px + i];
    const double PNr = (nb.jN == j) ? m.rp[gj] * pp[pc] : m.rm[gj + 1] * pp[nb.jN * s.px + i];
    a[pc] = a0;
    a[np + pc] = mm_Au(ub, za[2 * np + pc], pp[j * s.px + nb.iW], pp[j * s.px + nb.iE], dtt, dtcz);
    a[2 * np + pc] = mm_Av(lam1[s.poff + 2 * np + pc], ub, za[np + pc], PSr, PNr, dtf, dtt, m.dtcm);
}

// lam0 on the extended tile (contributions that land in ghost cells are dropped: perturbations
// of frozen ghost data are zero, R14)
__global__ void gk_adjL0(const Sub* __restrict__ subs, const int* __restrict__ mask, int n, ModelP m,
                         const double* __restrict__ Zp, const double* __restrict__ A,
                         double* __restrict__ lam0)
{
    GK_PROLOGUE
    if (n >= s.W || !is_interior(r, i, j)) return;
    const double* z = Zp + s.poff;
    const double* a = A + s.poff;
    double* l0 = lam0 + s.poff;
    const Nb nb = nbrs(r, i, j);
    const int gj = r.joff + j;
    const long long np = s.npad;
    const double dtcz = m.dtcz[gj], dtcm = m.dtcm;
    const int cE = j * s.px + nb.iE, cW = j * s.px + nb.iW, cN = nb.jN * s.px + i, cS = nb.jS * s.px + i;
    const double cuW = dtcz * z[np + cW], cuE = dtcz * z[np + cE];
    // mirrored pole row: v0 changes sign
    const double cvS = dtcm * nb.sS * z[2 * np + cS], cvN = dtcm * nb.sN * z[2 * np + cN];
    double out[3], su = 0.0, sv = 0.0;
#pragma unroll
    for (int f = 0; f < DD_NF; ++f) {
        const double* af = a + f * np;
        const double* zf = z + f * np;
        const double mN = f == 2 ? nb.sN : 1.0, mS = f == 2 ? nb.sS : 1.0;
        out[f] = mm_L0(af[pc], af[cW], af[cE], mS * af[cS], mN * af[cN], cuW, cuE, cvS, cvN, m.kap);
        su += (zf[cE] - zf[cW]) * af[pc];
        sv += (mN * zf[cN] - mS * zf[cS]) * af[pc];
    }
    l0[pc] = out[0];
    l0[np + pc] = out[1] - dtcz * su;
    l0[2 * np + pc] = out[2] - dtcm * sv;
}

// ------------------------------------------------------------------------------------------
// adjoint variable at the window end: the successor-window overlap forcing, eq (25c) case 2
// (R12): 2 mu (Z^{s_{j+1}} - x_{j+1,i}) / sigma_b^2, else zero.  Written into the
// buffer whose parity the sweep reaches at this subdomain's own window length.
__global__ void gk_adj_init(const Sub* __restrict__ subs, const int* __restrict__ mask, int Wmax,
                            int q, int p12, CostP cp, const double* __restrict__ traj,
                            const double* __restrict__ xfrozen, double* __restrict__ lamA,
                            double* __restrict__ lamB)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.ncell) return;
    double* lam = (((Wmax - s.W) & 1) ? lamB : lamA) + s.poff;
    const int lj = c / s.ex, li = c - lj * s.ex;
    const int pc = (lj + s.gys) * s.px + li + s.gx;
    const bool succ = s.jw < q - 1;
    const double* tw = traj + s.toff + (long long)s.W * DD_NF * s.ncell;
    const double* xn = succ ? xfrozen + subs[k + p12].coff : nullptr;
#pragma unroll
    for (int f = 0; f < DD_NF; ++f) {
        double v = 0.0;
        if (succ) v = 2.0 * cp.mu * (tw[(long long)f * s.ncell + c] - xn[(long long)f * s.ncell + c]) * cp.ib[f];
        lam[(long long)f * s.npad + pc] = v;
    }
}

// H^T R^-1 (misfit) at local level n added to the adjoint variable, eq (25b); obs are unique per
// (level, cell, field) inside a subdomain, so no atomics.
__global__ void gk_obs_force(const Sub* __restrict__ subs, const int* __restrict__ mask, int n,
                             const long long* __restrict__ obs_start, const int* __restrict__ obs_idx,
                             const double* __restrict__ obs_y, const double* __restrict__ obs_c,
                             const double* __restrict__ traj, double* __restrict__ lam)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    if (n > s.W) return;
    const long long q0 = obs_start[s.ooff + n], q1 = obs_start[s.ooff + n + 1];
    const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
    double* l = lam + s.poff;
    for (long long q = q0 + blockIdx.x * blockDim.x + threadIdx.x; q < q1; q += (long long)gridDim.x * blockDim.x) {
        const int idx = obs_idx[q];
        const int f = idx / s.ncell, c = idx - f * s.ncell;
        const int lj = c / s.ex, li = c - lj * s.ex;
        const double rr = t[idx] - obs_y[q];
        l[(long long)f * s.npad + (lj + s.gys) * s.px + li + s.gx] += 2.0 * obs_c[q] * rr;
    }
}

// ------------------------------------------------------------------------------------------
// Option overlap_levels: the spatial overlap penalty (25c) case 1 on EVERY level of the window
// (eq (21) l.300 read literally), generic path only.  ovl: the neighbours' frozen trajectories on the overlap
// rectangles, [W][3][novl] per subdomain (levels 1 .. W), refreshed by xk_ovl_fill at every exchange.
// Adjoint forcing at local level n >= 1: gather form (every cell looks up the rectangles that hold it).
__global__ void gk_ovl_force(const Sub* __restrict__ subs, const NbRect* __restrict__ nbr, const int* __restrict__ mask,
                             int n, CostP cp, const double* __restrict__ traj, const double* __restrict__ ovl,
                             double* __restrict__ lam)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    if (n < 1 || n > s.W || s.novl == 0) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.ncell) return;
    const int lj = c / s.ex, li = c - lj * s.ex;
    const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
    const double* o = ovl + s.voff + (long long)(n - 1) * DD_NF * s.novl;
    double acc[3] = { 0.0, 0.0, 0.0 };
    for (int r = 0; r < s.nnb; ++r) {
        const NbRect nb = nbr[s.nb0 + r];
        const int di = li - nb.i0, dj = lj - nb.j0;
        if ((unsigned)di < (unsigned)nb.w && (unsigned)dj < (unsigned)nb.h) {
            const int e = nb.ooff + dj * nb.w + di;
#pragma unroll
            for (int f = 0; f < 3; ++f) acc[f] += 2.0 * cp.mu * (t[(long long)f * s.ncell + c] - o[(long long)f * s.novl + e]) * cp.ib[f];
        }
    }
    double* l = lam + s.poff;
#pragma unroll
    for (int f = 0; f < 3; ++f) l[(long long)f * s.npad + (lj + s.gys) * s.px + li + s.gx] += acc[f];
}
// its cost, added to the spatial-overlap part and to J_ji (one CTA per subdomain, fixed-order sums)
template <int NT>
__global__ void gk_ovl_cost(const Sub* __restrict__ subs, const NbRect* __restrict__ nbr, const int* __restrict__ mask,
                            CostP cp, const double* __restrict__ traj, const double* __restrict__ ovl,
                            double* __restrict__ parts, double* __restrict__ J)
{
    __shared__ double red[32];
    const int k = blockIdx.x;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    double acc = 0.0;
    for (int r = 0; r < s.nnb; ++r) {
        const NbRect nb = nbr[s.nb0 + r];
        const int ncr = nb.w * nb.h;
        for (int q = threadIdx.x; q < ncr * s.W; q += NT) {
            const int n = q / ncr + 1, e = q - (n - 1) * ncr;
            const int dj = e / nb.w, di = e - dj * nb.w;
            const int c = (nb.j0 + dj) * s.ex + nb.i0 + di;
            const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
            const double* o = ovl + s.voff + (long long)(n - 1) * DD_NF * s.novl + nb.ooff + e;
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double dv = t[(long long)f * s.ncell + c] - o[(long long)f * s.novl];
                acc += dv * dv * cp.ib[f];
            }
        }
    }
    acc = block_sum<NT>(acc, red);
    if (threadIdx.x == 0) { parts[k * 5 + 2] += cp.mu * acc; J[k] += cp.mu * acc; }
}

// ------------------------------------------------------------------------------------------
// cost terms of J_ji, eq (25) l.338-344: partial sums per (block, subdomain), fixed order.
// parts: [nsub][CB][5] = bg (25a), obs (25b), spatial overlap, predecessor, successor (25c).
template <int NT>
__global__ void gk_cost_partial(const Sub* __restrict__ subs, const int* __restrict__ mask, GeoP geo,
                                CostP cp, const double* __restrict__ x, const double* __restrict__ xbs,
                                const double* __restrict__ xfrozen, const double* __restrict__ pred_end,
                                const double* __restrict__ traj, const long long* __restrict__ obs_start,
                                const int* __restrict__ obs_idx, const double* __restrict__ obs_y,
                                const double* __restrict__ obs_c, double* __restrict__ partial)
{
    __shared__ double sh[32];
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const int CB = gridDim.x;
    double bg = 0, ob = 0, sp = 0, pr = 0, su = 0;
    const int p12 = geo.p1 * geo.p2;
    const bool pred = s.jw > 0, succ = s.jw < geo.q - 1;
    const double* xk = x + s.coff;
    const double* xb = xbs + s.coff;
    const double* pe = pred_end + s.coff;
    const double* xn = succ ? xfrozen + subs[k + p12].coff : nullptr;
    const double* tw = traj + s.toff + (long long)s.W * DD_NF * s.ncell;
    for (int c = blockIdx.x * NT + threadIdx.x; c < s.ncell; c += CB * NT) {
        const int lj = c / s.ex, li = c - lj * s.ex;
        const int gi = imodd(s.ei0 + li, geo.nlon), gj = s.ej0 + lj;
        const int nc = geo.ncolcov[gi], nr = geo.nrowcov[gj];
        const double wsp = 1.0 / (double)(nc * nr);
#pragma unroll
        for (int f = 0; f < DD_NF; ++f) {
            const double xv = xk[(long long)f * s.ncell + c];
            const double db = xv - xb[(long long)f * s.ncell + c];
            bg += (s.jw == 0 ? 1.0 : cp.bgw) * wsp * db * db * cp.ib[f];
            if (nc * nr > 1)
                for (int cb = 0; cb < nr; ++cb)
                    for (int ca = 0; ca < nc; ++ca) {
                        const int a2 = geo.colcov[4 * gi + ca], b2 = geo.rowcov[4 * gj + cb];
                        if (a2 == s.a && b2 == s.b) continue;
                        const Sub& s2 = subs[(s.jw * geo.p2 + b2) * geo.p1 + a2];
                        const int li2 = imodd(gi - s2.ei0, geo.nlon), lj2 = gj - s2.ej0;
                        const double dv = xv - xfrozen[s2.coff + (long long)f * s2.ncell + lj2 * s2.ex + li2];
                        sp += dv * dv * cp.ib[f];
                    }
            if (pred) { const double dv = xv - pe[(long long)f * s.ncell + c]; pr += dv * dv * cp.ib[f]; }
            if (succ) {
                const double dv = tw[(long long)f * s.ncell + c] - xn[(long long)f * s.ncell + c];
                su += dv * dv * cp.ib[f];
            }
        }
    }
    if (obs_start) {
        const long long q0 = obs_start[s.ooff], q1 = obs_start[s.ooff + s.W + 1];
        // level of an observation = the bin it sits in; walk bins so that traj level is known
        for (int n = 0; n <= s.W; ++n) {
            const long long a0 = obs_start[s.ooff + n], a1 = obs_start[s.ooff + n + 1];
            const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
            for (long long q = a0 + blockIdx.x * NT + threadIdx.x; q < a1; q += (long long)CB * NT) {
                const double rr = t[obs_idx[q]] - obs_y[q];
                ob += obs_c[q] * rr * rr;
            }
        }
        (void)q0; (void)q1;
    }
    double v[5] = { bg, ob, cp.mu * sp, cp.mu * pr, cp.mu * su };
#pragma unroll
    for (int q = 0; q < 5; ++q) {
        const double t = block_sum<NT>(v[q], sh);
        if (threadIdx.x == 0) partial[((long long)k * CB + blockIdx.x) * 5 + q] = t;
    }
}
// parts[k][0..4] and J[k] = their sum (eq (25)); one thread per subdomain
__global__ void gk_cost_final(int nsub, const int* __restrict__ mask, int CB,
                              const double* __restrict__ partial, double* __restrict__ parts,
                              double* __restrict__ J)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nsub || (mask && !mask[k])) return;
    double tot = 0.0;
    for (int q = 0; q < 5; ++q) {
        double v = 0.0;
        for (int b = 0; b < CB; ++b) v += partial[((long long)k * CB + b) * 5 + q];
        parts[k * 5 + q] = v;
        tot += v;
    }
    J[k] = tot;
}

// gradient at the window start: adjoint variable + (25a) + control-level (25c) terms; also the
// gradient in the B-preconditioned variable w (eq (44) l.630-634): g_w = sigma_b g_x.
__global__ void gk_grad_final(const Sub* __restrict__ subs, const int* __restrict__ mask, GeoP geo,
                              CostP cp, const double* __restrict__ x, const double* __restrict__ xbs,
                              const double* __restrict__ xfrozen, const double* __restrict__ pred_end,
                              const double* __restrict__ lam, double* __restrict__ gx,
                              double* __restrict__ gw)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.ncell) return;
    const int lj = c / s.ex, li = c - lj * s.ex;
    const int gi = imodd(s.ei0 + li, geo.nlon), gj = s.ej0 + lj;
    const int nc = geo.ncolcov[gi], nr = geo.nrowcov[gj];
    const double wsp = 1.0 / (double)(nc * nr);
    const int pc = (lj + s.gys) * s.px + li + s.gx;
    const bool pred = s.jw > 0;
#pragma unroll
    for (int f = 0; f < DD_NF; ++f) {
        const long long o = s.coff + (long long)f * s.ncell + c;
        const double xv = x[o];
        double g = lam[s.poff + (long long)f * s.npad + pc];
        g += 2.0 * (s.jw == 0 ? 1.0 : cp.bgw) * wsp * (xv - xbs[o]) * cp.ib[f];
        if (nc * nr > 1)
            for (int cb = 0; cb < nr; ++cb)
                for (int ca = 0; ca < nc; ++ca) {
                    const int a2 = geo.colcov[4 * gi + ca], b2 = geo.rowcov[4 * gj + cb];
                    if (a2 == s.a && b2 == s.b) continue;
                    const Sub& s2 = subs[(s.jw * geo.p2 + b2) * geo.p1 + a2];
                    const int li2 = imodd(gi - s2.ei0, geo.nlon), lj2 = gj - s2.ej0;
                    g += 2.0 * cp.mu * (xv - xfrozen[s2.coff + (long long)f * s2.ncell + lj2 * s2.ex + li2]) * cp.ib[f];
                }
        if (pred) g += 2.0 * cp.mu * (xv - pred_end[o]) * cp.ib[f];
        if (gx) gx[o] = g;
        if (gw) gw[o] = cp.sb[f] * g;
    }
}
