// cost_kernels.cuh -- the control-level terms of the local functional J_ji (eq (25) l.338-344) for the
// wavefront sweep kernels (wave_forward.cuh / wave_adjoint.cuh), one CTA per subdomain.
//
// wk_forward leaves the trajectory store.  Every term of J_ji is evaluated here from data in global memory, in
// one bandwidth-bound pass over the control plus the sparse samples of the trajectory at the observations:
//   (25a) background term, weight 1/multiplicity (R6, R7)
//   (25b) misfits, cost and the forcing 2 c (H Z^n - y) of the adjoint sweep (obs_r) at every level of the window
//   (25c) spatial overlap with the frozen controls of the neighbour tiles (gather form: every cell
//         looks up the rectangles that contain it), predecessor window, successor window (Z^W)
// and, for the adjoint sweep that follows,
//   gx   := gradient of the control-level terms (wk_adjoint adds lambda^0 with reductions)
//   lamW := 2 mu (Z^W - x_succ) / sigma_b^2 (zero in the last window) + the observation forcing of level W: the adjoint
//           variable at the window end
//   level 0 of the trajectory store := the control.
// Sums: per thread in cell order, then the fixed tree of block_sum: no atomics, run-to-run identical.
#pragma once
#include "wave_common.cuh"

#define CK_NT 256

__global__ void __launch_bounds__(CK_NT, 5) ck_cost(const WkArgs A)
{
    __shared__ double red[32];
    const int k = blockIdx.x, tid = threadIdx.x;
    if (A.mask && !A.mask[k]) return;
    const Sub s = A.subs[k];
    const int nc = s.ncell;
    const bool pred = s.jw > 0, succ = s.jw < A.geo.q - 1;
    const double bw = s.jw == 0 ? 1.0 : A.cp.bgw;
    const double mu2 = 2.0 * A.cp.mu;
    const double* x = A.x + s.coff;
    const double* xb = A.xbs + s.coff;
    const double* pe = A.pred_end + s.coff;
    const double* zw = A.traj + s.toff + (long long)s.W * 3 * nc;
    const double* xn = succ ? A.xfrozen + A.subs[k + A.geo.p1 * A.geo.p2].coff : nullptr;
    double* t0 = A.traj + s.toff;
    double* gx = A.gx + s.coff;
    double* lw = A.lamW + s.coff;
    double bg = 0.0, sp = 0.0, pr = 0.0, su = 0.0, ob = 0.0;
    for (int c = tid; c < nc; c += CK_NT) {
        const int lj = c / s.ex, li = c - lj * s.ex;
        int gi = s.ei0 + li; gi = gi < 0 ? gi + A.geo.nlon : (gi >= A.geo.nlon ? gi - A.geo.nlon : gi);
        const double wsp = bw / (double)(A.geo.ncolcov[gi] * A.geo.nrowcov[s.ej0 + lj]);
        double xv[3], gv[3];
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            xv[f] = __ldg(x + (long long)f * nc + c);
            const double db = xv[f] - __ldg(xb + (long long)f * nc + c);
            bg += wsp * db * db * A.cp.ib[f];
            gv[f] = 2.0 * wsp * db * A.cp.ib[f];
            if (pred) {
                const double dv = xv[f] - __ldg(pe + (long long)f * nc + c);
                pr += dv * dv * A.cp.ib[f];
                gv[f] += mu2 * dv * A.cp.ib[f];
            }
            double lv = 0.0;
            if (succ) {
                const double dv = __ldg(zw + (long long)f * nc + c) - __ldg(xn + (long long)f * nc + c);
                su += dv * dv * A.cp.ib[f];
                lv = mu2 * dv * A.cp.ib[f];
            }
            lw[(long long)f * nc + c] = lv;
            t0[(long long)f * nc + c] = xv[f];
        }
        // (25c) case 1: one rectangle per (neighbour tile, periodic image) of the same window
        for (int r = 0; r < s.nnb; ++r) {
            const NbRect nb = A.nbr[s.nb0 + r];
            const int di = li - nb.i0, dj = lj - nb.j0;
            if ((unsigned)di < (unsigned)nb.w && (unsigned)dj < (unsigned)nb.h) {
                const double* xf = A.xfrozen + nb.coff2 + (long long)(nb.nj0 + dj) * nb.ex2 + nb.ni0 + di;
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    const double dv = xv[f] - __ldg(xf + (long long)f * nb.ncell2);
                    sp += dv * dv * A.cp.ib[f];
                    gv[f] += mu2 * dv * A.cp.ib[f];
                }
            }
        }
#pragma unroll
        for (int f = 0; f < 3; ++f) gx[(long long)f * nc + c] = gv[f];
    }
    __syncthreads();                            // gx of every cell is in place (global writes of this CTA)
    // H (25b) at level 0: misfit, cost, and its gradient straight into gx (cells are unique inside a level, R20)
    if (A.obs_start) {
        const long long a0 = A.obs_start[s.ooff], a1 = A.obs_start[s.ooff + 1];
        for (long long q = a0 + tid; q < a1; q += CK_NT) {
            const int pk = A.obs_lj[q];
            const long long o = (long long)((pk >> 8) & 3) * nc + (pk >> 12) * s.ex + (pk & 255);
            const double rr = __ldg(x + o) - A.obs_y[q];
            const double cq = A.obs_c[q];
            ob += cq * rr * rr;
            const double r2 = 2.0 * cq * rr;
            A.obs_r[q] = r2;
            gx[o] += r2;
        }
    }
    // H (25b) at the levels 1 .. W: sampled from the trajectory store the forward sweep has just written
    if (A.obs_start) {
        for (int n = 1; n <= s.W; ++n) {
            const long long a0 = A.obs_start[s.ooff + n], a1 = A.obs_start[s.ooff + n + 1];
            const double* tn = A.traj + s.toff + (long long)n * 3 * nc;
            for (long long q = a0 + tid; q < a1; q += CK_NT) {
                const int pk = A.obs_lj[q];
                const double rr = tn[(long long)((pk >> 8) & 3) * nc + (pk >> 12) * s.ex + (pk & 255)] - A.obs_y[q];
                const double cq = A.obs_c[q];
                ob += cq * rr * rr;
                const double r2 = 2.0 * cq * rr;
                A.obs_r[q] = r2;
                // the forcing of level W goes straight into lambda^W (unique cells inside a level; the __syncthreads above
                // ordered the writes of lamW): the first adjoint step of the window then carries no observation work
                if (n == s.W) lw[(long long)((pk >> 8) & 3) * nc + (pk >> 12) * s.ex + (pk & 255)] += r2;
            }
        }
    }
    bg = block_sum<CK_NT>(bg, red);
    sp = block_sum<CK_NT>(sp, red);
    pr = block_sum<CK_NT>(pr, red);
    su = block_sum<CK_NT>(su, red);
    ob = block_sum<CK_NT>(ob, red);
    if (tid == 0) {
        const double v[5] = { bg, ob, A.cp.mu * sp, A.cp.mu * pr, A.cp.mu * su };
        double tot = 0.0;
        for (int q = 0; q < 5; ++q) { A.parts[k * 5 + q] = v[q]; tot += v[q]; }
        A.J[k] = tot;
    }
}

// g_w = sigma_b g_x (eq (44) l.630-634): the gradient the L-BFGS of a5 works with
__global__ void ck_scale_grad(const Sub* __restrict__ subs, const int* __restrict__ mask, CostP cp,
                              const double* __restrict__ gx, double* __restrict__ gw)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < 3 * s.ncell; c += gridDim.x * blockDim.x)
        gw[s.coff + c] = cp.sb[c / s.ncell] * gx[s.coff + c];
}
