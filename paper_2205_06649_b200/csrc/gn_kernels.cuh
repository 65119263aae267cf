// gn_kernels.cuh -- the paper's own local minimiser: incremental Gauss-Newton on J_ji
// (Algorithm 5 l.568-589, Algorithm 6 l.655-685) with the normal equations (42)-(43) l.620-626 solved by
// conjugate gradients in w = V^+ (u - u^b), V = diag(sigma_b) (eq (44)-(46) l.630-649, the "B-preconditioned"
// system of Algorithm 7 l.688-696; R21), batched over all subdomains.
//
// One product with H_GN = 2 grad F^T grad F (F = the stacked residuals of eq (25) l.338-344):
//   tk_init    dZ^0 = V p on the padded tile, zero on the frozen ghost ring
//   tk_step    dZ^{n+1} = M_n dZ^n, the tangent-linear model about the stored trajectory (TLM, Alg 6 l.14-16);
//              one launch per step, a CTA computes a 32x16 tile in shared memory (overlapped tiling, the
//              non-linear intermediates h^a, u^a, v^a, h^1, u^1 recomputed beside their perturbations)
//   tk_obs     2 c H dZ^{n+1}: the forcing of the adjoint sweep at an observation level (25b)
//   ck_gn      control-level terms 2 (w (25a) + mu (25c)) dx / sigma_b^2, level-0 observations, and
//              lambda^W = 2 mu dZ^W / sigma_b^2 (successor window)
//   wk_adjoint the adjoint sweep (ADJ, Alg 6 l.17-19), unchanged: it linearises about the same trajectory
// and the CG recurrences per subdomain (one CTA each, fixed-order block sums: run-to-run identical).
#pragma once
#include "common.cuh"
#include "generic_kernels.cuh"
#include "model_math.cuh"
#include "step_kernels.cuh"
#include "wave_common.cuh"

#define TK_SMEM_DOUBLES (6 * (SK_TY + 6) * (SK_TX + 6) + 6 * (SK_TY + 4) * (SK_TX + 4) + 2 * (SK_TY + 2) * (SK_TX + 2))

// dZ^0: interior = sigma_b p (p in w-space, control layout), ghost ring = 0; both ping-pong buffers' rings are cleared
__global__ void tk_init(const Sub* __restrict__ subs, CostP cp, const double* __restrict__ pw,
                        double* __restrict__ dA, double* __restrict__ dB)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    const Reg r = make_reg(s);
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.npad) return;
    const int j = c / s.px, i = c - j * s.px;
    const bool in = is_interior(r, i, j);
#pragma unroll
    for (int f = 0; f < 3; ++f) {
        const long long o = s.poff + (long long)f * s.npad + c;
        if (in) dA[o] = cp.sb[f] * pw[s.coff + (long long)f * s.ncell + (j - s.gys) * s.ex + (i - s.gx)];
        else { dA[o] = 0.0; dB[o] = 0.0; }
    }
}

// TLM of step n on one 32x16 output tile: din / dout padded [3][npad] arrays (zero on the ghost ring)
__global__ void __launch_bounds__(SK_NT) tk_step(const Sub* __restrict__ subs, int n, ModelP m,
                                                 const double* __restrict__ traj, const double* __restrict__ ghost,
                                                 const double* __restrict__ din, double* __restrict__ dout, int tiles_x)
{
    constexpr int W0 = SK_TX + 6, H0 = SK_TY + 6, W1 = SK_TX + 4, H1 = SK_TY + 4, W2 = SK_TX + 2, H2 = SK_TY + 2;
    extern __shared__ double tk_sm[];
    double* z0 = tk_sm;                       // [3][H0*W0]
    double* d0 = z0 + 3 * H0 * W0;            // [3][H0*W0]
    double* za = d0 + 3 * H0 * W0;            // [3][H1*W1]
    double* da = za + 3 * H1 * W1;            // [3][H1*W1]
    double* h1 = da + 3 * H1 * W1;            // [H2*W2]
    double* dh = h1 + H2 * W2;                // [H2*W2]
    const int k = blockIdx.y;
    const Sub s = subs[k];
    if (n >= s.W) return;
    const Reg r = make_reg(s);
    const int tx = blockIdx.x % tiles_x, ty = blockIdx.x / tiles_x;
    const int oi = s.gx + tx * SK_TX, oj = s.gys + ty * SK_TY;
    if (oi >= s.gx + s.ex || oj >= s.gys + s.ey) return;
    const double* t = traj + s.toff + (long long)n * DD_NF * s.ncell;
    const double* g = ghost + s.goff + (long long)n * DD_NF * s.nring;
    const double* di = din + s.poff;
    const long long np = s.npad;
    for (int c = threadIdx.x; c < H0 * W0; c += SK_NT) {
        const int lj = c / W0, li = c - lj * W0;
        const int i = oi - 3 + li, j = oj - 3 + lj;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0, e0 = 0.0, e1 = 0.0, e2 = 0.0;
        if (sk_inside(r, i, j)) {
            const int iw = sk_wrap(r, i);
            v0 = sk_z0(s, r, t, g, 0, iw, j); v1 = sk_z0(s, r, t, g, 1, iw, j); v2 = sk_z0(s, r, t, g, 2, iw, j);
            const int pc = j * s.px + iw;
            e0 = di[pc]; e1 = di[np + pc]; e2 = di[2 * np + pc];
        }
        z0[c] = v0; z0[H0 * W0 + c] = v1; z0[2 * H0 * W0 + c] = v2;
        d0[c] = e0; d0[H0 * W0 + c] = e1; d0[2 * H0 * W0 + c] = e2;
    }
    __syncthreads();
    // ---- stage A and its TLM on the tile + 2 (range 1)
    for (int c = threadIdx.x; c < H1 * W1; c += SK_NT) {
        const int lj = c / W1, li = c - lj * W1;
        const int i = oi - 2 + li, j = oj - 2 + lj;
        double a[3] = { 0.0, 0.0, 0.0 }, b[3] = { 0.0, 0.0, 0.0 };
        if (sk_range(r, 1, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int cc = (lj + 1) * W0 + li + 1, cN = (jN - oj + 3) * W0 + li + 1, cS = (jS - oj + 3) * W0 + li + 1;
            const double dtcz = m.dtcz[r.joff + j];
            const double cu = dtcz * z0[H0 * W0 + cc], cv = m.dtcm * z0[2 * H0 * W0 + cc];
            const double dcu = dtcz * d0[H0 * W0 + cc], dcv = m.dtcm * d0[2 * H0 * W0 + cc];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double* zf = z0 + f * H0 * W0; const double* df = d0 + f * H0 * W0;
                const double mN = f == 2 ? sN : 1.0, mS = f == 2 ? sS : 1.0;
                const double xE = zf[cc + 1], xW = zf[cc - 1], xN = mN * zf[cN], xS = mS * zf[cS];
                const double yE = df[cc + 1], yW = df[cc - 1], yN = mN * df[cN], yS = mS * df[cS];
                a[f] = mm_stageA(zf[cc], xE, xW, xN, xS, cu, cv, m.kap);
                // d(x^a) = dx - [dcu (xE - xW) + cu (dxE - dxW) + dcv (xN - xS) + cv (dxN - dxS)] + kappa L(dx)
                b[f] = df[cc] - (dcu * (xE - xW) + cu * (yE - yW) + dcv * (xN - xS) + cv * (yN - yS)) +
                       m.kap * (yE + yW + yN + yS - 4.0 * df[cc]);
            }
        }
        za[c] = a[0]; za[H1 * W1 + c] = a[1]; za[2 * H1 * W1 + c] = a[2];
        da[c] = b[0]; da[H1 * W1 + c] = b[1]; da[2 * H1 * W1 + c] = b[2];
    }
    __syncthreads();
    // ---- h^1 and dh^1 on the tile + 1 (range 2)
    for (int c = threadIdx.x; c < H2 * W2; c += SK_NT) {
        const int lj = c / W2, li = c - lj * W2;
        const int i = oi - 1 + li, j = oj - 1 + lj;
        double v = 0.0, dv = 0.0;
        if (sk_range(r, 2, i, j)) {
            int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
            const int cc = (lj + 1) * W1 + li + 1, cN = (jN - oj + 2) * W1 + li + 1, cS = (jS - oj + 2) * W1 + li + 1;
            const int gj = r.joff + j;
            const double* ua = za + H1 * W1; const double* va = za + 2 * H1 * W1;
            const double* dua = da + H1 * W1; const double* dva = da + 2 * H1 * W1;
            const double D = mm_div(ua[cc + 1], ua[cc - 1], sN * va[cN], sS * va[cS], m.dtcz[gj], m.dtcm, m.rp[gj], m.rm[gj]);
            const double dD = mm_div(dua[cc + 1], dua[cc - 1], sN * dva[cN], sS * dva[cS], m.dtcz[gj], m.dtcm, m.rp[gj], m.rm[gj]);
            v = mm_h1(za[cc], D);
            dv = da[cc] - (da[cc] * D + za[cc] * dD);         // d(h^a - h^a D)
        }
        h1[c] = v; dh[c] = dv;
    }
    __syncthreads();
    // ---- du^1, dv^1 on the tile -> dout (extended-tile cells only)
    double* dn = dout + s.poff;
    for (int c = threadIdx.x; c < SK_TY * SK_TX; c += SK_NT) {
        const int lj = c / SK_TX, li = c - lj * SK_TX;
        const int i = oi + li, j = oj + lj;
        if (i >= s.gx + s.ex || j >= s.gys + s.ey) continue;
        int jN, jS; double sN, sS; sk_ns(r, j, jN, jS, sN, sS);
        const int ca = (lj + 2) * W1 + li + 2;
        const int ch = (lj + 1) * W2 + li + 1, chN = (jN - oj + 1) * W2 + li + 1, chS = (jS - oj + 1) * W2 + li + 1;
        const int gj = r.joff + j;
        const double dtf = m.dtf[gj], dtt = m.dtt[gj];
        const double ua = za[H1 * W1 + ca], va = za[2 * H1 * W1 + ca];
        const double dua = da[H1 * W1 + ca], dva = da[2 * H1 * W1 + ca];
        const double u1 = mm_u1(ua, va, h1[ch + 1], h1[ch - 1], m.gdtcz[gj], dtf, dtt);
        // d(u^a - gdtcz (h1E - h1W) + (dtf + dtt u^a) v^a)
        const double du1 = dua - m.gdtcz[gj] * (dh[ch + 1] - dh[ch - 1]) + dtt * dua * va + (dtf + dtt * ua) * dva;
        // d(v^a - gdtcm (h1N - h1S) - (dtf + dtt u^1) u^1)
        const double dv1 = dva - m.gdtcm * (dh[chN] - dh[chS]) - (dtf + 2.0 * dtt * u1) * du1;
        const int pc = j * s.px + i;
        dn[pc] = dh[ch]; dn[np + pc] = du1; dn[2 * np + pc] = dv1;
    }
}

// generic layouts: level lev of the tangent-linear trajectory, padded array -> trajectory-store layout [(W+1)][3][ncell]
__global__ void tk_store(const Sub* __restrict__ subs, int lev, const double* __restrict__ dz, double* __restrict__ dtraj)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    if (lev > s.W) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= s.ncell) return;
    const int lj = c / s.ex, li = c - lj * s.ex;
    const int pc = (lj + s.gys) * s.px + li + s.gx;
#pragma unroll
    for (int f = 0; f < 3; ++f)
        dtraj[s.toff + ((long long)lev * 3 + f) * s.ncell + c] = dz[s.poff + (long long)f * s.npad + pc];
}

// forcing of the adjoint sweep at local level lev: rt[q] = 2 c (H dZ^lev)[q]  (c = lambda w / sigma_o^2, eq (25b))
__global__ void tk_obs(const Sub* __restrict__ subs, int lev, const long long* __restrict__ obs_start,
                       const int* __restrict__ obs_lj, const double* __restrict__ obs_c,
                       const double* __restrict__ dz, double* __restrict__ rt)
{
    const int k = blockIdx.y;
    const Sub s = subs[k];
    if (lev > s.W) return;
    const long long a0 = obs_start[s.ooff + lev], a1 = obs_start[s.ooff + lev + 1];
    for (long long q = a0 + blockIdx.x * blockDim.x + threadIdx.x; q < a1; q += (long long)gridDim.x * blockDim.x) {
        const int pk = obs_lj[q];
        const int f = (pk >> 8) & 3, lj = pk >> 12, li = pk & 255;
        rt[q] = 2.0 * obs_c[q] * dz[s.poff + (long long)f * s.npad + (lj + s.gys) * s.px + li + s.gx];
    }
}

// control-level part of H_GN p (x-space, before the final sigma_b): one CTA per subdomain.
// dA / dB: the ping-pong TLM buffers; dZ^W sits in dA when W is even.
__global__ void __launch_bounds__(256) ck_gn(const Sub* __restrict__ subs, const NbRect* __restrict__ nbr, GeoP geo, CostP cp,
                                              const double* __restrict__ pw, const double* __restrict__ dA,
                                              const double* __restrict__ dB, const long long* __restrict__ obs_start,
                                              const int* __restrict__ obs_lj, const double* __restrict__ obs_c,
                                              double* __restrict__ rt, double* __restrict__ gxh, double* __restrict__ lamW)
{
    const int k = blockIdx.x, tid = threadIdx.x;
    const Sub s = subs[k];
    const int nc = s.ncell;
    const bool pred = s.jw > 0, succ = s.jw < geo.q - 1;
    const double bw = s.jw == 0 ? 1.0 : cp.bgw, mu2 = 2.0 * cp.mu;
    const double* dW = ((s.W & 1) ? dB : dA) + s.poff;
    for (int c = tid; c < nc; c += 256) {
        const int lj = c / s.ex, li = c - lj * s.ex;
        int gi = s.ei0 + li; gi = gi < 0 ? gi + geo.nlon : (gi >= geo.nlon ? gi - geo.nlon : gi);
        const double wsp = bw / (double)(geo.ncolcov[gi] * geo.nrowcov[s.ej0 + lj]);
        int nr = 0;                             // number of neighbour tiles (images) whose extended tile holds the cell
        for (int r = 0; r < s.nnb; ++r) {
            const NbRect nb = nbr[s.nb0 + r];
            if ((unsigned)(li - nb.i0) < (unsigned)nb.w && (unsigned)(lj - nb.j0) < (unsigned)nb.h) ++nr;
        }
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            const long long o = s.coff + (long long)f * nc + c;
            const double dx = cp.sb[f] * pw[o];
            double gv = 2.0 * wsp * dx * cp.ib[f];
            for (int r = 0; r < nr; ++r) gv += mu2 * dx * cp.ib[f];
            if (pred) gv += mu2 * dx * cp.ib[f];
            gxh[o] = gv;
            lamW[o] = succ ? mu2 * dW[(long long)f * s.npad + (lj + s.gys) * s.px + li + s.gx] * cp.ib[f] : 0.0;
        }
    }
    __syncthreads();
    if (obs_start) {                            // (25b) at level 0
        const long long a0 = obs_start[s.ooff], a1 = obs_start[s.ooff + 1];
        for (long long q = a0 + tid; q < a1; q += 256) {
            const int pk = obs_lj[q];
            const long long o = s.coff + (long long)((pk >> 8) & 3) * nc + (pk >> 12) * s.ex + (pk & 255);
            const double r2 = 2.0 * obs_c[q] * cp.sb[(pk >> 8) & 3] * pw[o];
            rt[q] = r2;
            gxh[o] += r2;
        }
        // level W: the forcing tk_obs left in rt goes into lambda^W (wk_adjoint carries no observation work at level W)
        const long long b0 = obs_start[s.ooff + s.W], b1 = obs_start[s.ooff + s.W + 1];
        for (long long q = b0 + tid; q < b1; q += 256) {
            const int pk = obs_lj[q];
            lamW[s.coff + (long long)((pk >> 8) & 3) * nc + (pk >> 12) * s.ex + (pk & 255)] += rt[q];
        }
    }
}

// dx = sigma_b p (x-space perturbation of the control)
__global__ void gn_scale_x(const Sub* __restrict__ subs, CostP cp, const double* __restrict__ pw, double* __restrict__ dx)
{
    const Sub s = subs[blockIdx.y];
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < 3 * s.ncell; c += gridDim.x * blockDim.x)
        dx[s.coff + c] = cp.sb[c / s.ncell] * pw[s.coff + c];
}

// ---- conjugate gradients on H_GN dw = -g, one CTA per subdomain; vectors in control layout [3][ncell]
#define GN_NT 512
__global__ void __launch_bounds__(GN_NT) gn_cg_init(const Sub* __restrict__ subs, const double* __restrict__ g,
                                                    double* __restrict__ dw, double* __restrict__ rv,
                                                    double* __restrict__ pv, double* __restrict__ rr, int* __restrict__ stop)
{
    __shared__ double red[32];
    const int k = blockIdx.x;
    const Sub s = subs[k];
    double acc = 0.0;
    for (int c = threadIdx.x; c < 3 * s.ncell; c += GN_NT) {
        const long long o = s.coff + c;
        const double r = -g[o];
        dw[o] = 0.0; rv[o] = r; pv[o] = r;
        acc += r * r;
    }
    acc = block_sum<GN_NT>(acc, red);
    if (threadIdx.x == 0) { rr[k] = acc; stop[k] = acc > 0.0 ? 0 : 1; }
}
__global__ void __launch_bounds__(GN_NT) gn_cg_update(const Sub* __restrict__ subs, const double* __restrict__ Hp,
                                                      double* __restrict__ dw, double* __restrict__ rv,
                                                      double* __restrict__ pv, double* __restrict__ rr, int* __restrict__ stop)
{
    __shared__ double red[32];
    const int k = blockIdx.x;
    if (stop[k]) return;
    const Sub s = subs[k];
    const int n = 3 * s.ncell;
    double acc = 0.0;
    for (int c = threadIdx.x; c < n; c += GN_NT) acc += pv[s.coff + c] * Hp[s.coff + c];
    const double pHp = block_sum<GN_NT>(acc, red);
    if (!(pHp > 0.0)) { if (threadIdx.x == 0) stop[k] = 1; return; }
    const double rr0 = rr[k], al = rr0 / pHp;
    acc = 0.0;
    for (int c = threadIdx.x; c < n; c += GN_NT) {
        const long long o = s.coff + c;
        dw[o] += al * pv[o];
        const double r = rv[o] - al * Hp[o];
        rv[o] = r;
        acc += r * r;
    }
    const double rr2 = block_sum<GN_NT>(acc, red);
    const double be = rr2 / rr0;
    for (int c = threadIdx.x; c < n; c += GN_NT) {
        const long long o = s.coff + c;
        pv[o] = rv[o] + be * pv[o];
    }
    if (threadIdx.x == 0) { rr[k] = rr2; if (!(rr2 > 0.0)) stop[k] = 1; }
}
__global__ void gn_add(const Sub* __restrict__ subs, double* __restrict__ w, const double* __restrict__ dw)
{
    const Sub s = subs[blockIdx.y];
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < 3 * s.ncell; c += gridDim.x * blockDim.x)
        w[s.coff + c] += dw[s.coff + c];
}
