// exchange_kernels.cuh -- Algorithm 1 l.465 "Exchange u_ji between adjacent subdomains" and
// l.470 "Gather", all inside device memory: refresh of the frozen ghost-ring trajectories,
// predecessor end states and frozen controls, the step norm (l.466), the restriction of a
// global state to the tiles (Def 4 l.164-170) and the weighted extension-sum (eq (12)-(13)
// l.194-201).
#pragma once
#include "common.cuh"
#include "model_math.cuh"

// ghost[k][n][f][r] <- traj[owner][n][f][cell]: every ghost cell takes the value of the tile
// that OWNS it, same window, all levels that start a step (R14).
__global__ void xk_ghost_fill(const Sub* __restrict__ subs, GeoP geo, const double* __restrict__ traj,
                              double* __restrict__ ghost)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    const int rr = blockIdx.x * blockDim.x + threadIdx.x;
    if (rr >= s.nring) return;
    // ring index -> padded coordinates (inverse of the enumeration in gk_fill_pad)
    int i, j;
    const int nsouth = s.gys * s.px, nns = (s.gys + s.gyn) * s.px;
    if (rr < nsouth) { j = rr / s.px; i = rr - j * s.px; }
    else if (rr < nns) { const int q = rr - nsouth; j = s.gys + s.ey + q / s.px; i = q % s.px; }
    else {
        const int q = rr - nns, w2 = 2 * s.gx;
        const int lj = q / w2, t = q - lj * w2;
        j = s.gys + lj; i = t < s.gx ? t : t + s.ex;
    }
    const int gi = imodd(s.ei0 - s.gx + i, geo.nlon), gj = s.ej0 - s.gys + j;
    const Sub& so = subs[(s.jw * geo.p2 + geo.rowown[gj]) * geo.p1 + geo.colown[gi]];
    const int li = imodd(gi - so.ei0, geo.nlon), lj = gj - so.ej0;
    const long long c = (long long)lj * so.ex + li;
    for (int n = blockIdx.z; n < s.W; n += gridDim.z) {
        const double* t = traj + so.toff + (long long)n * DD_NF * so.ncell;
        double* g = ghost + s.goff + (long long)n * DD_NF * s.nring;
#pragma unroll
        for (int f = 0; f < DD_NF; ++f) g[(long long)f * s.nring + rr] = t[(long long)f * so.ncell + c];
    }
}

// pred_end[k] <- final state of the predecessor window on the same tile (eq (25c) case 2);
// delta_k = ||x_k - xfrozen_k||_inf (l.466, l.704); xfrozen[k] <- x[k].
template <int NT>
__global__ void xk_freeze(const Sub* __restrict__ subs, GeoP geo, const double* __restrict__ traj,
                          const double* __restrict__ x, double* __restrict__ xfrozen,
                          double* __restrict__ pred_end, double* __restrict__ dmax, const int* __restrict__ own)
{
    // own (sharded runs, dd4dvar_set_owned_windows): this process freezes the controls of the subdomains it owns and
    // the end states of the windows it owns (= pred_end of their successors); the rest is imported from the owners
    __shared__ double sh[32];
    const int k = blockIdx.x;
    const Sub s = subs[k];
    const int n3 = DD_NF * s.ncell;
    const bool mine = !own || own[k];
    double mx = 0.0;
    const double* tp = nullptr;
    if (s.jw > 0 && (!own || own[k - geo.p1 * geo.p2])) {
        const Sub& sp = subs[k - geo.p1 * geo.p2];
        tp = traj + sp.toff + (long long)sp.W * DD_NF * sp.ncell;
    }
    for (int q = threadIdx.x; q < n3; q += NT) {
        if (mine) {
            const double xn = x[s.coff + q];
            mx = fmax(mx, fabs(xn - xfrozen[s.coff + q]));
            xfrozen[s.coff + q] = xn;
        }
        if (tp) pred_end[s.coff + q] = tp[q];
    }
    mx = block_max<NT>(mx, sh);
    if (threadIdx.x == 0 && mine) dmax[k] = mx;
}

// traj[k][n] <- restriction of global level s_k + n (source = the undecomposed layout's store)
__global__ void xk_restrict_level(const Sub* __restrict__ subs, int nlon, int nlat, int level,
                                  const double* __restrict__ gstate, double* __restrict__ traj,
                                  double* __restrict__ xbs, double* __restrict__ x)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    if (level < s.s || level > s.s + s.W) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.ncell) return;
    const int lj = c / s.ex, li = c - lj * s.ex;
    const int gi = imodd(s.ei0 + li, nlon), gj = s.ej0 + lj;
    double* t = traj + s.toff + (long long)(level - s.s) * DD_NF * s.ncell;
#pragma unroll
    for (int f = 0; f < DD_NF; ++f) {
        const double v = gstate[((long long)f * nlat + gj) * nlon + gi];
        t[(long long)f * s.ncell + c] = v;
        if (level == s.s) { xbs[s.coff + (long long)f * s.ncell + c] = v; x[s.coff + (long long)f * s.ncell + c] = v; }
    }
}

// out[f][gj][gi] = sum over the subdomains that hold (level, cell) of weight * value, in
// ascending subdomain order; weight = 1/multiplicity (Def 4 generalised, R6).
// mode 0: from the trajectory store at `level`; mode 1: analysis = window-0 frozen controls.
__global__ void xk_gather(const Sub* __restrict__ subs, GeoP geo, int mode, int level,
                          const double* __restrict__ src, double* __restrict__ out)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= geo.nlon * geo.nlat) return;
    const int gj = g / geo.nlon, gi = g - gj * geo.nlon;
    const int nc = geo.ncolcov[gi], nr = geo.nrowcov[gj];
    int jw0 = 0, jw1 = 0, tm = 1;
    if (mode == 0) {
        jw0 = -1;
        for (int jw = 0; jw < geo.q; ++jw)
            if (level >= geo.wb[jw] && level <= geo.wb[jw + 1]) { if (jw0 < 0) jw0 = jw; jw1 = jw; }
        tm = jw1 - jw0 + 1;
    }
    const double wt = 1.0 / (double)(nc * nr) / (double)tm;
    const double wsp = 1.0 / (double)(nc * nr);
    double acc[3] = { 0.0, 0.0, 0.0 };
    for (int jw = jw0; jw <= jw1; ++jw)
        for (int cb = 0; cb < nr; ++cb)
            for (int ca = 0; ca < nc; ++ca) {
                const Sub& s = subs[(jw * geo.p2 + geo.rowcov[4 * gj + cb]) * geo.p1 + geo.colcov[4 * gi + ca]];
                const int li = imodd(gi - s.ei0, geo.nlon), lj = gj - s.ej0;
                const long long c = (long long)lj * s.ex + li;
                const double* p = mode == 0 ? src + s.toff + (long long)(level - s.s) * DD_NF * s.ncell
                                            : src + s.coff;
#pragma unroll
                for (int f = 0; f < DD_NF; ++f)
                    acc[f] += (mode == 0 ? wt : wsp) * p[(long long)f * s.ncell + c];
            }
#pragma unroll
    for (int f = 0; f < DD_NF; ++f) out[((long long)f * geo.nlat + gj) * geo.nlon + gi] = acc[f];
}

// Frozen boundary data derived from the ghost ring (wavefront kernels, wave_common.cuh): the
// stage-A value u^a (R3; eq (61) l.948-951 advective part) in the ghost columns 1 and
// px-2 of every padded row and every level that starts a step.  It depends on ghost cells only
// (columns 0..2 resp. px-3..px-1, rows r-1..r+1), so it changes with the exchange, not with the
// control.  Layout per (subdomain, level): [S rows gys][N rows gyn][tile rows ey] x {west, east}.
__global__ void xk_edge_ua(const Sub* __restrict__ subs, ModelP m, const double* __restrict__ ghost,
                           double* __restrict__ gedge)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= 2 * s.py) return;
    const int r = q >> 1, side = q & 1;
    const int c = side ? s.px - 2 : 1;
    const bool ws = s.gys == 0, wn = s.gyn == 0;
    const int gj = s.ej0 - s.gys + r;
    const double dtcz = m.dtcz[gj < 0 ? 0 : (gj >= m.nlat ? m.nlat - 1 : gj)];
    int slot;                                   // position of padded row r in the layout above
    if (r < s.gys) slot = r;
    else if (r >= s.gys + s.ey) slot = s.gys + (r - s.gys - s.ey);
    else slot = s.gys + s.gyn + (r - s.gys);
    for (int n = blockIdx.z; n < s.W; n += gridDim.z) {
        const double* gz = ghost + s.goff + (long long)n * DD_NF * s.nring;
        auto G = [&](int f, int rr, int cc) -> double {
            const double* p = gz + (long long)f * s.nring;
            if (rr < s.gys) return p[rr * s.px + cc];
            if (rr >= s.gys + s.ey) return p[s.gys * s.px + (rr - s.gys - s.ey) * s.px + cc];
            return p[(s.gys + s.gyn) * s.px + (rr - s.gys) * 2 * s.gx + (cc < s.gx ? cc : cc - s.ex)];
        };
        // north / south neighbours: the mirrored edge row at a pole wall (u is even under the mirror);
        // on an open side rows 0 and py-1 lie outside the range of stage A and are never used
        const int rN = r + 1 < s.py ? r + 1 : r, rS = r > 0 ? r - 1 : r;
        (void)ws; (void)wn;
        const double u = G(1, r, c), v = G(2, r, c);
        const double ua = mm_stageA(u, G(1, r, c + 1), G(1, r, c - 1), G(1, rN, c), G(1, rS, c), dtcz * u, m.dtcm * v, m.kap);
        gedge[s.eoff + (long long)n * 2 * s.py + slot * 2 + side] = ua;
    }
}

// Option overlap_levels: the neighbours' trajectories of this iteration on the overlap rectangles, levels 1 .. W
// (same window, same local level), into the compact overlap store [W][3][novl] of every subdomain.
__global__ void xk_ovl_fill(const Sub* __restrict__ subs, const NbRect* __restrict__ nbr,
                            const double* __restrict__ traj, double* __restrict__ ovl)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= s.novl) return;
    int r = 0;
    while (r + 1 < s.nnb && nbr[s.nb0 + r + 1].ooff <= e) ++r;
    const NbRect nb = nbr[s.nb0 + r];
    const int q = e - nb.ooff, dj = q / nb.w, di = q - dj * nb.w;
    const long long c2 = (long long)(nb.nj0 + dj) * nb.ex2 + nb.ni0 + di;
    for (int n = 1 + blockIdx.z; n <= s.W; n += gridDim.z)
#pragma unroll
        for (int f = 0; f < DD_NF; ++f)
            ovl[s.voff + ((long long)(n - 1) * DD_NF + f) * s.novl + e] =
                traj[nb.toff2 + ((long long)n * DD_NF + f) * nb.ncell2 + c2];
}
