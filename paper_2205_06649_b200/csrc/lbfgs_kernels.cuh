// lbfgs_kernels.cuh -- batched per-subdomain L-BFGS (Liu-Nocedal two-loop recursion; PAPER.md
// Remark 3 l.595, l.941 refs [29],[11]) in the B-preconditioned variable w = (x - u^b(s_j)) /
// sigma_b (eq (44) l.630-634).  Constants and branch rules: DESIGN.md R10.  One CTA per
// subdomain; all reductions are fixed-order block sums, so results do not depend on scheduling.
#pragma once
#include "common.cuh"

struct LbfgsP {
    int m, max_bt;
    double c1;
    long long ctot;      // length of one control-shaped array (stride between history slots)
};
// per-subdomain optimiser state (device arrays of length nsub unless noted)
struct LbfgsState {
    double* J;       // cost at the current iterate
    double* Jt;      // cost at the trial point
    double* t;       // trial step
    double* gd;      // g.d
    int* nh;         // pairs stored
    int* head;       // ring start (oldest pair)
    int* active;     // line search still running
    int* ok;         // line search accepted a trial
    int* done;       // zero gradient: subdomain finished for this outer iteration
    int* trial;      // halvings so far
    double* rho;     // [nsub][m]
    double* gam;     // [nsub][m]  s.y / y.y of the pair in that slot
    int* nactive;    // [1] counter
};

template <int NT>
__device__ __forceinline__ double bdot(const double* __restrict__ a, const double* __restrict__ b, int n,
                                       double* sh)
{
    double v = 0.0;
    for (int q = threadIdx.x; q < n; q += NT) v += a[q] * b[q];
    return block_sum<NT>(v, sh);
}

// search direction d = -H g by the two-loop recursion with H0 = (s'y / y'y) I; empty history (or
// a non-descent direction): d = -g with trial step 1/||g||.
template <int NT>
__global__ void __launch_bounds__(NT) lk_direction(const Sub* __restrict__ subs, LbfgsP lp, LbfgsState st,
                                                   const double* __restrict__ g, const double* __restrict__ S,
                                                   const double* __restrict__ Y, double* __restrict__ d)
{
    __shared__ double sh[32];
    __shared__ double alpha[32];
    const int k = blockIdx.x;
    const Sub s = subs[k];
    if (st.done[k]) { if (threadIdx.x == 0) { st.active[k] = 0; st.ok[k] = 0; } return; }
    const int n = DD_NF * s.ncell;
    const double* gk = g + s.coff;
    double* dk = d + s.coff;
    const double gg = bdot<NT>(gk, gk, n, sh);
    const double gnorm = sqrt(gg);
    if (!(gnorm > 0.0)) {
        if (threadIdx.x == 0) { st.done[k] = 1; st.active[k] = 0; st.ok[k] = 0; }
        return;
    }
    int nh = st.nh[k];
    const int head = st.head[k];
    double t0 = 1.0, gd = 0.0;
    if (nh > 0) {
        for (int q = threadIdx.x; q < n; q += NT) dk[q] = gk[q];
        __syncthreads();
        for (int i = nh - 1; i >= 0; --i) {
            const int slot = (head + i) % lp.m;
            const double* si = S + (long long)slot * lp.ctot + s.coff;
            const double* yi = Y + (long long)slot * lp.ctot + s.coff;
            const double al = st.rho[k * lp.m + slot] * bdot<NT>(si, dk, n, sh);
            if (threadIdx.x == 0) alpha[i] = al;
            for (int q = threadIdx.x; q < n; q += NT) dk[q] -= al * yi[q];
            __syncthreads();
        }
        const double gamma = st.gam[k * lp.m + (head + nh - 1) % lp.m];
        for (int q = threadIdx.x; q < n; q += NT) dk[q] *= gamma;
        __syncthreads();
        for (int i = 0; i < nh; ++i) {
            const int slot = (head + i) % lp.m;
            const double* si = S + (long long)slot * lp.ctot + s.coff;
            const double* yi = Y + (long long)slot * lp.ctot + s.coff;
            const double beta = st.rho[k * lp.m + slot] * bdot<NT>(yi, dk, n, sh);
            const double co = alpha[i] - beta;
            for (int q = threadIdx.x; q < n; q += NT) dk[q] += si[q] * co;
            __syncthreads();
        }
        for (int q = threadIdx.x; q < n; q += NT) dk[q] = -dk[q];
        __syncthreads();
        gd = bdot<NT>(gk, dk, n, sh);
        if (!(gd < 0.0)) nh = 0;   // not a descent direction: restart
    }
    if (nh == 0) {
        for (int q = threadIdx.x; q < n; q += NT) dk[q] = -gk[q];
        t0 = 1.0 / gnorm;
        gd = -(gnorm * gnorm);
    }
    if (threadIdx.x == 0) {
        st.nh[k] = nh; if (nh == 0) st.head[k] = 0;
        st.t[k] = t0; st.gd[k] = gd; st.trial[k] = 0; st.active[k] = 1; st.ok[k] = 0;
    }
}

// trial point wt = w + t d and the physical control x = u^b(s_j) + sigma_b wt
__global__ void lk_trial(const Sub* __restrict__ subs, const int* __restrict__ mask, CostP cp,
                         const double* __restrict__ tstep, const double* __restrict__ w,
                         const double* __restrict__ d, const double* __restrict__ xbs,
                         double* __restrict__ wt, double* __restrict__ x)
{
    const int k = blockIdx.y;
    if (mask && !mask[k]) return;
    const Sub s = subs[k];
    const double t = tstep ? tstep[k] : 0.0;
    const int n = DD_NF * s.ncell;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += gridDim.x * blockDim.x) {
        const int f = q / s.ncell;
        const long long o = s.coff + q;
        const double wv = d ? w[o] + t * d[o] : w[o];
        if (wt) wt[o] = wv;
        x[o] = xbs[o] + cp.sb[f] * wv;
    }
}

// Armijo test J(w + t d) <= J + c1 t g.d; otherwise halve, up to max_bt halvings
__global__ void lk_lscheck(int nsub, LbfgsP lp, LbfgsState st)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nsub || !st.active[k]) return;
    const double t = st.t[k];
    if (st.Jt[k] <= st.J[k] + lp.c1 * t * st.gd[k]) { st.ok[k] = 1; st.active[k] = 0; return; }
    const int b = st.trial[k] + 1;
    if (b > lp.max_bt) { st.active[k] = 0; st.ok[k] = 0; return; }
    st.trial[k] = b;
    st.t[k] = 0.5 * t;
    atomicAdd(st.nactive, 1);
}

// accepted step: new pair (s, y) = (wt - w, gn - g), kept if s'y > 1e-12 ||s|| ||y||; oldest pair
// dropped when the history is full; w <- wt, g <- gn, J <- Jt.  Rejected line search: history
// cleared, iterate kept.
template <int NT>
__global__ void __launch_bounds__(NT) lk_update(const Sub* __restrict__ subs, LbfgsP lp, LbfgsState st,
                                                double* __restrict__ w, const double* __restrict__ wt,
                                                double* __restrict__ g, const double* __restrict__ gn,
                                                double* __restrict__ S, double* __restrict__ Y)
{
    __shared__ double sh[32];
    const int k = blockIdx.x;
    if (st.done[k]) return;
    const Sub s = subs[k];
    if (!st.ok[k]) { if (threadIdx.x == 0) { st.nh[k] = 0; st.head[k] = 0; } return; }
    const int n = DD_NF * s.ncell;
    double* wk = w + s.coff; const double* wtk = wt + s.coff;
    double* gk = g + s.coff; const double* gnk = gn + s.coff;
    if (lp.m > 0) {
        int nh = st.nh[k], head = st.head[k];
        if (nh == lp.m) { head = (head + 1) % lp.m; nh = lp.m - 1; }
        const int slot = (head + nh) % lp.m;
        double* sn = S + (long long)slot * lp.ctot + s.coff;
        double* yn = Y + (long long)slot * lp.ctot + s.coff;
        double sy = 0.0, ss = 0.0, yy = 0.0;
        for (int q = threadIdx.x; q < n; q += NT) {
            const double sv = wtk[q] - wk[q], yv = gnk[q] - gk[q];
            sn[q] = sv; yn[q] = yv;
            sy += sv * yv; ss += sv * sv; yy += yv * yv;
        }
        sy = block_sum<NT>(sy, sh); ss = block_sum<NT>(ss, sh); yy = block_sum<NT>(yy, sh);
        if (sy > 1e-12 * sqrt(ss) * sqrt(yy)) {
            if (threadIdx.x == 0) { st.rho[k * lp.m + slot] = 1.0 / sy; st.gam[k * lp.m + slot] = sy / yy; }
            ++nh;
        }
        if (threadIdx.x == 0) { st.nh[k] = nh; st.head[k] = head; }
    }
    for (int q = threadIdx.x; q < n; q += NT) { wk[q] = wtk[q]; gk[q] = gnk[q]; }
    if (threadIdx.x == 0) st.J[k] = st.Jt[k];
}
