// fused_forward.cuh -- the forward row-marching kernel with static register slots (see
// fused_adjoint.cuh for the conventions: tick loop unrolled by 4, histories indexed by row & 3,
// virtual mirrored pole rows, branch-free steady ticks, persistent CTAs over a work counter).
// The current state of the window lives IN PLACE in this CTA's slot of the L2-pinned scratch (row j
// of level n+1 overwrites row j of level n three ticks after the same thread read it), so HBM only
// sees the trajectory store being written (streaming stores) and the frozen ghost ring being read.
// (included once per CTA width from fused_kernels.cuh, inside a namespace; FK_NT = threads per CTA)

struct FwdRegs {
    double z[4][3];
    double ha[2], ua[4], va[4], h1[4];
    double zq[3];     // row t+2 in flight
};
struct FwdCtx {
    FkGeo g;
    int cj;                         // joff + 1: index of padded row 0 in the row tables
    const double* tb;               // this handle's row tables [6][FK_CTAB]
    FkCol col;
    double* z0s;      // [2][3][FK_NT]
    double* uas;      // [2][FK_NT]
    double* h1s;      // [2][FK_NT]
    double* scol;     // this thread's column of the in-place state
    double* tcol;     // this thread's column of trajectory level n+1
    int nc1, gys, ex, py;
    double kap, dtcm, gdtcm;
};

template <int PH, bool ST>
__device__ __forceinline__ void fwd_tick(const int t, FwdRegs& R, const FwdCtx& C)
{
#define SL(lag) ((PH - (lag)) & 3)
#define S2(lag) ((PH - (lag)) & 1)
    const FkGeo& g = C.g;
    const int i = g.i;
    // ---- S0: row t has arrived; request row t+1; publish row t
    if (!ST && t == C.py && g.wn) { R.z[SL(0)][0] = R.z[SL(1)][0]; R.z[SL(0)][1] = R.z[SL(1)][1]; R.z[SL(0)][2] = -R.z[SL(1)][2]; }
    R.z[SL(-1)][0] = R.zq[0]; R.z[SL(-1)][1] = R.zq[1]; R.z[SL(-1)][2] = R.zq[2];     // row t+1 (requested at t-1)
    if (ST || t + 2 < C.py) fk_load_row(g, C.col, t + 2, R.zq);
    if (ST || t < C.py) {
        double* zw = C.z0s + (S2(0) * 3) * FK_NT + i;
        zw[0] = R.z[SL(0)][0]; zw[FK_NT] = R.z[SL(0)][1]; zw[2 * FK_NT] = R.z[SL(0)][2];
        if (!ST && t == 0 && g.ws) { R.z[SL(1)][0] = R.z[SL(0)][0]; R.z[SL(1)][1] = R.z[SL(0)][1]; R.z[SL(1)][2] = -R.z[SL(0)][2]; }
    }
    // ---- S1: stage A on row j = t-1
    {
        const int j = t - 1;
        if (ST || (j >= g.jA0 && j < g.jA1)) {
            const double* zc = R.z[SL(1)];
            const double cu = ctab(CT_DTCZ, C.cj, j) * zc[1], cv = C.dtcm * zc[2];
            const double* zE = C.z0s + (S2(1) * 3) * FK_NT + g.iE;
            const double* zW = C.z0s + (S2(1) * 3) * FK_NT + g.iW;
            R.ha[S2(1)] = mm_stageA(zc[0], zE[0], zW[0], R.z[SL(0)][0], R.z[SL(2)][0], cu, cv, C.kap);
            const double ua = mm_stageA(zc[1], zE[FK_NT], zW[FK_NT], R.z[SL(0)][1], R.z[SL(2)][1], cu, cv, C.kap);
            R.va[SL(1)] = mm_stageA(zc[2], zE[2 * FK_NT], zW[2 * FK_NT], R.z[SL(0)][2], R.z[SL(2)][2], cu, cv, C.kap);
            R.ua[SL(1)] = ua;
            C.uas[S2(1) * FK_NT + i] = ua;
            if (!ST && j == 0 && g.ws) R.va[SL(2)] = -R.va[SL(1)];
        } else if (!ST && j == C.py && g.wn) R.va[SL(1)] = -R.va[SL(2)];
    }
    // ---- S2: h1 on row j = t-2
    {
        const int j = t - 2;
        if (ST || (j >= g.jH0 && j < g.jH1)) {
            const double D = mm_div(C.uas[S2(2) * FK_NT + g.iE], C.uas[S2(2) * FK_NT + g.iW], R.va[SL(1)], R.va[SL(3)],
                                    ctab(CT_DTCZ, C.cj, j), C.dtcm, ctab(CT_RP, C.cj, j), ctab(CT_RM, C.cj, j));
            const double h1 = mm_h1(R.ha[S2(2)], D);
            R.h1[SL(2)] = h1;
            C.h1s[S2(2) * FK_NT + i] = h1;
            if (!ST && j == 0 && g.ws) R.h1[SL(3)] = h1;
        } else if (!ST && j == C.py && g.wn) R.h1[SL(2)] = R.h1[SL(3)];
    }
    // ---- S3: u1, v1 on row j = t-3 -> trajectory store (streaming) and in-place state
    {
        const int j = t - 3;
        if (ST || (j >= g.jU0 && j < g.jU1)) {
            const double dtf = ctab(CT_DTF, C.cj, j), dtt = ctab(CT_DTT, C.cj, j);
            const double u1 = mm_u1(R.ua[SL(3)], R.va[SL(3)], C.h1s[S2(3) * FK_NT + g.iE], C.h1s[S2(3) * FK_NT + g.iW],
                                    ctab(CT_GDTCZ, C.cj, j), dtf, dtt);
            const double v1 = mm_v1(R.va[SL(3)], u1, R.h1[SL(2)], R.h1[SL(4)], C.gdtcm, dtf, dtt);
            if (g.cU) {
                const int o = (j - C.gys) * C.ex;
                const double h1 = R.h1[SL(3)];
                __stcs(C.tcol + o, h1); __stcs(C.tcol + C.nc1 + o, u1); __stcs(C.tcol + 2 * C.nc1 + o, v1);
                C.scol[o] = h1; C.scol[C.nc1 + o] = u1; C.scol[2 * C.nc1 + o] = v1;
            }
        }
    }
#undef SL
#undef S2
}

__global__ void __launch_bounds__(FK_NT, 512 / FK_NT) fk_forward2(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                        ModelP m, const double* __restrict__ x, double* traj,
                                                        const double* ghost, int nsub, double* scratch,
                                                        long long slot_stride, int* counter,
                                                        const double* __restrict__ ctabp)
{
    __shared__ double z0s[2 * 3 * FK_NT];
    __shared__ double uas[2 * FK_NT];
    __shared__ double h1s[2 * FK_NT];
    __shared__ int s_next;
    for (;;) {
        if (threadIdx.x == 0) s_next = atomicAdd(counter, 1);
        __syncthreads();
        const int k = s_next;
        __syncthreads();
        if (k >= nsub) break;
        if (mask && !mask[k]) continue;
        const Sub s = subs[k];
        FwdCtx C;
        C.g = fk_geo(s);
        C.cj = C.g.joff + 1;
        C.tb = ctabp;
        const FkGeo& g = C.g;
        double* state = scratch + (long long)blockIdx.x * slot_stride;
        C.z0s = z0s; C.uas = uas; C.h1s = h1s;
        C.nc1 = s.ncell; C.gys = s.gys; C.ex = s.ex; C.py = s.py;
        C.kap = m.kap; C.dtcm = m.dtcm; C.gdtcm = m.gdtcm;
        C.scol = state + (g.cU ? g.li : 0);
        // level 0 of the store = the control; it is also the initial in-place state
        for (int c = threadIdx.x; c < 3 * s.ncell; c += FK_NT) {
            const double v = x[s.coff + c];
            state[c] = v;
            __stcs(traj + s.toff + c, v);
        }
        __syncthreads();
        const int T = (s.py + 3 + 3) & ~3;
        const int ts0 = (g.jU0 + 3 + 3) & ~3, ts1 = s.py - 3;
        for (int n = 0; n < s.W; ++n) {
            C.tcol = traj + s.toff + (long long)(n + 1) * 3 * s.ncell + (g.cU ? g.li : 0);
            C.col = fk_col(g, state, ghost + s.goff + (long long)n * 3 * s.nring);
            FwdRegs R;
#pragma unroll
            for (int q = 0; q < 4; ++q) { R.z[q][0] = R.z[q][1] = R.z[q][2] = 0.0; R.ua[q] = R.va[q] = R.h1[q] = 0.0; }
            R.ha[0] = R.ha[1] = 0.0;
            fk_load_row(g, C.col, 0, R.z[0]);
            R.zq[0] = R.zq[1] = R.zq[2] = 0.0;
            if (s.py > 1) fk_load_row(g, C.col, 1, R.zq);
            for (int t0 = 0; t0 < T; t0 += 4) {
                if (t0 >= ts0 && t0 + 3 <= ts1) {
                    fwd_tick<0, true>(t0, R, C); __syncthreads();
                    fwd_tick<1, true>(t0 + 1, R, C); __syncthreads();
                    fwd_tick<2, true>(t0 + 2, R, C); __syncthreads();
                    fwd_tick<3, true>(t0 + 3, R, C); __syncthreads();
                } else {
                    fwd_tick<0, false>(t0, R, C); __syncthreads();
                    fwd_tick<1, false>(t0 + 1, R, C); __syncthreads();
                    fwd_tick<2, false>(t0 + 2, R, C); __syncthreads();
                    fwd_tick<3, false>(t0 + 3, R, C); __syncthreads();
                }
            }
        }
    }
}
