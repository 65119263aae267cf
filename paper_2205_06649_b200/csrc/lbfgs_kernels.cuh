// lbfgs_kernels.cuh -- batched per-subdomain L-BFGS (Liu-Nocedal two-loop recursion; PAPER.md
// Remark 3 l.595, l.941 refs [29],[11]) in the B-preconditioned variable w = (x - u^b(s_j)) /
// sigma_b (eq (44) l.630-634).  Constants and branch rules: DESIGN.md R10.  One thread-block
// CLUSTER (LK_CL CTAs) per subdomain: each CTA owns a strided share of the vectors, dot products
// are fixed-order block sums exchanged through distributed shared memory and added in rank order,
// so results do not depend on scheduling and every CTA of the cluster takes the same branches.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
namespace cg = cooperative_groups;

#define LK_CL 4      // CTAs per cluster = per subdomain

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
    int* nactive;    // [0] counter of subdomains still searching, [1] non-finite-gradient flag
};

// Sum over the whole cluster (= over the whole subdomain vector) of per-thread partial sums:
// fixed-order block sum in every CTA, partials exchanged through distributed shared memory and
// added in cluster-rank order, so every CTA holds the same bit pattern.  `slot` alternates between
// two exchange buffers so that one cluster.sync per reduction is enough.
template <int NT>
__device__ __forceinline__ double cluster_sum(double v, double* sh /*[32]*/, double* xch /*[2]*/, int& slot)
{
    cg::cluster_group cl = cg::this_cluster();
    const double part = block_sum<NT>(v, sh);
    if (threadIdx.x == 0) xch[slot] = part;
    cl.sync();
    double tot = 0.0;
    for (unsigned r = 0; r < cl.num_blocks(); ++r) tot += *cl.map_shared_rank(xch + slot, r);
    slot ^= 1;
    return tot;
}
// element range of this thread inside the subdomain vector: q = q0, q0 + stride, ...
#define LK_FOR(q, n) for (int q = (int)cg::this_cluster().block_rank() * NT + (int)threadIdx.x; q < (n); q += LK_CL * NT)

template <int NT>
__device__ __forceinline__ double cdot(const double* __restrict__ a, const double* __restrict__ b, int n,
                                       double* sh, double* xch, int& slot)
{
    double v = 0.0;
    LK_FOR(q, n) v += a[q] * b[q];
    return cluster_sum<NT>(v, sh, xch, slot);
}

// search direction d = -H g by the two-loop recursion with H0 = (s'y / y'y) I; empty history (or
// a non-descent direction): d = -g with trial step 1/||g||.
template <int NT>
__global__ void __cluster_dims__(LK_CL, 1, 1) __launch_bounds__(NT) lk_direction(const Sub* __restrict__ subs, LbfgsP lp, LbfgsState st,
                                                   const double* __restrict__ g, const double* __restrict__ S,
                                                   const double* __restrict__ Y, double* __restrict__ d)
{
    __shared__ double sh[32];
    __shared__ double alpha[32];
    __shared__ double xch[2];
    cg::cluster_group cl = cg::this_cluster();
    const bool lead = cl.block_rank() == 0 && threadIdx.x == 0;
    int xs = 0;
    const int k = blockIdx.x / LK_CL;
    const Sub s = subs[k];
    // all state is read before the first cluster barrier; the leader writes it after the last one
    const int done = st.done[k];
    int nh = st.nh[k];
    const int head = st.head[k];
    if (done) { if (lead) { st.active[k] = 0; st.ok[k] = 0; } return; }
    const int n = DD_NF * s.ncell;
    const double* gk = g + s.coff;
    double* dk = d + s.coff;
    const double gg = cdot<NT>(gk, gk, n, sh, xch, xs);
    const double gnorm = sqrt(gg);
    if (!(gnorm > 0.0) || isinf(gnorm)) {
        // zero gradient: converged.  NaN / Inf gradient: frozen too, but reported (nactive[1] -> run returns -5)
        if (lead) { st.done[k] = 1; st.active[k] = 0; st.ok[k] = 0; if (!(gnorm == 0.0)) atomicExch(st.nactive + 1, 1); }
        cl.sync();
        return;
    }
    double t0 = 1.0, gd = 0.0;
    if (nh > 0) {
        // every thread owns the same elements of d in every loop: no barrier between the passes
        LK_FOR(q, n) dk[q] = gk[q];
        for (int i = nh - 1; i >= 0; --i) {
            const int slot = (head + i) % lp.m;
            const double* si = S + (long long)slot * lp.ctot + s.coff;
            const double* yi = Y + (long long)slot * lp.ctot + s.coff;
            const double al = st.rho[k * lp.m + slot] * cdot<NT>(si, dk, n, sh, xch, xs);
            if (threadIdx.x == 0) alpha[i] = al;
            LK_FOR(q, n) dk[q] -= al * yi[q];
        }
        __syncthreads();
        const double gamma = st.gam[k * lp.m + (head + nh - 1) % lp.m];
        LK_FOR(q, n) dk[q] *= gamma;
        for (int i = 0; i < nh; ++i) {
            const int slot = (head + i) % lp.m;
            const double* si = S + (long long)slot * lp.ctot + s.coff;
            const double* yi = Y + (long long)slot * lp.ctot + s.coff;
            const double beta = st.rho[k * lp.m + slot] * cdot<NT>(yi, dk, n, sh, xch, xs);
            const double co = alpha[i] - beta;
            LK_FOR(q, n) dk[q] += si[q] * co;
        }
        LK_FOR(q, n) dk[q] = -dk[q];
        gd = cdot<NT>(gk, dk, n, sh, xch, xs);
        if (!(gd < 0.0)) nh = 0;   // not a descent direction: restart
    }
    if (nh == 0) {
        LK_FOR(q, n) dk[q] = -gk[q];
        t0 = 1.0 / gnorm;
        gd = -(gnorm * gnorm);
    }
    if (lead) {
        st.nh[k] = nh; if (nh == 0) st.head[k] = 0;
        st.t[k] = t0; st.gd[k] = gd; st.trial[k] = 0; st.active[k] = 1; st.ok[k] = 0;
    }
    cl.sync();      // no CTA leaves while its exchange buffer may still be read
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
__global__ void __cluster_dims__(LK_CL, 1, 1) __launch_bounds__(NT) lk_update(const Sub* __restrict__ subs, LbfgsP lp, LbfgsState st,
                                                double* __restrict__ w, const double* __restrict__ wt,
                                                double* __restrict__ g, const double* __restrict__ gn,
                                                double* __restrict__ S, double* __restrict__ Y)
{
    __shared__ double sh[32];
    __shared__ double xch[2];
    cg::cluster_group cl = cg::this_cluster();
    const bool lead = cl.block_rank() == 0 && threadIdx.x == 0;
    int xs = 0;
    const int k = blockIdx.x / LK_CL;
    const int done = st.done[k], ok = st.ok[k];
    int nh = st.nh[k], head = st.head[k];
    if (done) return;
    const Sub s = subs[k];
    if (!ok) { if (lead) { st.nh[k] = 0; st.head[k] = 0; } return; }
    const int n = DD_NF * s.ncell;
    double* wk = w + s.coff; const double* wtk = wt + s.coff;
    double* gk = g + s.coff; const double* gnk = gn + s.coff;
    if (lp.m > 0) {
        if (nh == lp.m) { head = (head + 1) % lp.m; nh = lp.m - 1; }
        const int slot = (head + nh) % lp.m;
        double* sn = S + (long long)slot * lp.ctot + s.coff;
        double* yn = Y + (long long)slot * lp.ctot + s.coff;
        double sy = 0.0, ss = 0.0, yy = 0.0;
        LK_FOR(q, n) {
            const double sv = wtk[q] - wk[q], yv = gnk[q] - gk[q];
            sn[q] = sv; yn[q] = yv;
            sy += sv * yv; ss += sv * sv; yy += yv * yv;
        }
        sy = cluster_sum<NT>(sy, sh, xch, xs); ss = cluster_sum<NT>(ss, sh, xch, xs); yy = cluster_sum<NT>(yy, sh, xch, xs);
        if (sy > 1e-12 * sqrt(ss) * sqrt(yy)) {
            if (lead) { st.rho[k * lp.m + slot] = 1.0 / sy; st.gam[k * lp.m + slot] = sy / yy; }
            ++nh;
        }
        if (lead) { st.nh[k] = nh; st.head[k] = head; }
    }
    LK_FOR(q, n) { wk[q] = wtk[q]; gk[q] = gnk[q]; }
    if (lead) st.J[k] = st.Jt[k];
    cl.sync();
}
