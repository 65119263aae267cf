// fused_adjoint.cuh -- the adjoint row-marching kernel with STATIC register slots.
//
// Same pipeline as described in fused_kernels.cuh (adjoint tick t: load Z0[t] | stage A + UB row
// t-1 | HB,P row t-2 | A row t-3 | lam0 row t-4), but the tick loop is unrolled by 4 and every
// per-column history lives in a register array indexed by (row & 3) (or & 1), which is a
// compile-time constant inside each unrolled tick: no register rotation moves.  Reflective pole
// walls (R4) are handled by VIRTUAL rows -1 and py that hold the mirrored edge row
// (v-like quantities negated), written once per step under a uniform branch, so the stage code has
// no wall selects.  For P the mirror carries the metric ratio: P[-1] = r-_0 P[0], r+_{-1} := 1,
// P[py] = r+_{py-1} P[py-1], r-_{py} := 1 (see model_math.cuh, A_v).
// (included once per CTA width from fused_kernels.cuh, inside a namespace; FK_NT = threads per CTA)

struct AdjRegs {
    double z[4][3];                 // Z0 rows, slot = row & 3
    double ha[2], ua[4], va[4];     // stage A output
    double hb[2], vb[4], UB[4];     // adjoint variable at level n+1 (h, v) and UB
    double HB[2], P[4];
    double A[4][3];
    double l0, l1, l2, l3;          // prefetched lam row (h,u,v) and u1
};
struct AdjCtx {
    FkGeo g;
    int cj;                         // joff + 1: index of padded row 0 in the row tables
    const double* tb;               // this handle's row tables [6][FK_CTAB]
    FkCol col;
    double* zr;                     // [8][3][FK_NT]
    double* uas;                    // [4][FK_NT]
    double* ubs;                    // [2][FK_NT]
    double* ps;                     // [2][FK_NT]
    double* as;                     // [2][3][FK_NT]
    double* lcol;                   // this thread's column of lam
    const double* tu;               // this thread's column of u^1
    int nc1, gys, ex, py;
    double kap, dtcm, gdtcm, c0;
};

// slot of row (t - lag) in the 8-deep Z ring, t = t0 + PH, t0 % 4 == 0, h = t0 & 4
template <int PH, int LAG>
__device__ __forceinline__ int zr_slot(int h)
{
    constexpr int d = PH - LAG;
    constexpr int q = d >= 0 ? 0 : (d >= -4 ? -1 : -2);
    constexpr int r = d - 4 * q;
    return ((q & 1) ? (h ^ 4) : h) + r;
}

template <int PH, bool ST>
__device__ __forceinline__ void adj_tick(const int t, const int h, AdjRegs& R, const AdjCtx& C)
{
#define SL(lag) ((PH - (lag)) & 3)
#define S2(lag) ((PH - (lag)) & 1)
    const FkGeo& g = C.g;
    const int i = g.i;
    // ---- S0: row t of Z0 has arrived in its slot; request row t+1; publish row t
    if (!ST && t == C.py && g.wn) { R.z[SL(0)][0] = R.z[SL(1)][0]; R.z[SL(0)][1] = R.z[SL(1)][1]; R.z[SL(0)][2] = -R.z[SL(1)][2]; }
    if (ST || t + 1 < C.py) fk_load_row(g, C.col, t + 1, R.z[SL(-1)]);
    if (ST || t < C.py || (t == C.py && g.wn)) {
        double* zw = C.zr + (zr_slot<PH, 0>(h) * 3) * FK_NT + i;
        zw[0] = R.z[SL(0)][0]; zw[FK_NT] = R.z[SL(0)][1]; zw[2 * FK_NT] = R.z[SL(0)][2];
        if (!ST && t == 0 && g.ws) {     // virtual row -1 = mirrored row 0
            R.z[SL(1)][0] = R.z[SL(0)][0]; R.z[SL(1)][1] = R.z[SL(0)][1]; R.z[SL(1)][2] = -R.z[SL(0)][2];
            double* zv = C.zr + (7 * 3) * FK_NT + i;
            zv[0] = R.z[SL(0)][0]; zv[FK_NT] = R.z[SL(0)][1]; zv[2 * FK_NT] = -R.z[SL(0)][2];
        }
    }
    // ---- S1: stage A on row j = t-1
    {
        const int j = t - 1;
        if (ST || (j >= g.jA0 && j < g.jA1)) {
            const double* zc = R.z[SL(1)];
            const double cu = ctab(CT_DTCZ, C.cj, j) * zc[1], cv = C.dtcm * zc[2];
            const double* zE = C.zr + (zr_slot<PH, 1>(h) * 3) * FK_NT + g.iE;
            const double* zW = C.zr + (zr_slot<PH, 1>(h) * 3) * FK_NT + g.iW;
            R.ha[S2(1)] = mm_stageA(zc[0], zE[0], zW[0], R.z[SL(0)][0], R.z[SL(2)][0], cu, cv, C.kap);
            const double ua = mm_stageA(zc[1], zE[FK_NT], zW[FK_NT], R.z[SL(0)][1], R.z[SL(2)][1], cu, cv, C.kap);
            R.va[SL(1)] = mm_stageA(zc[2], zE[2 * FK_NT], zW[2 * FK_NT], R.z[SL(0)][2], R.z[SL(2)][2], cu, cv, C.kap);
            R.ua[SL(1)] = ua;
            C.uas[SL(1) * FK_NT + i] = ua;
            if (!ST && j == 0 && g.ws) R.va[SL(2)] = -R.va[SL(1)];
        } else if (!ST && j == C.py && g.wn) R.va[SL(1)] = -R.va[SL(2)];
        // lam row j (prefetched) -> hb, vb, UB (exact zeros outside the extended tile)
        double UB = 0.0, hb = 0.0, vb = 0.0;
        if (ST || (j >= g.jU0 && j < g.jU1)) {
            if (g.cU) { hb = R.l0; vb = R.l2; UB = mm_UB(R.l1, R.l2, R.l3, ctab(CT_DTF, C.cj, j), ctab(CT_DTT, C.cj, j)); }
            if (!ST && j == 0 && g.ws) R.vb[SL(2)] = -vb;
        } else if (!ST && j == C.py && g.wn) vb = -R.vb[SL(2)];
        R.hb[S2(1)] = hb; R.vb[SL(1)] = vb; R.UB[SL(1)] = UB;
        C.ubs[S2(1) * FK_NT + i] = UB;
        if (ST || (j + 1 >= g.jU0 && j + 1 < g.jU1)) {
            const int o = (j + 1 - C.gys) * C.ex;
            R.l0 = C.lcol[o]; R.l1 = C.lcol[C.nc1 + o]; R.l2 = C.lcol[2 * C.nc1 + o]; R.l3 = C.tu[o];
        }
    }
    // ---- S2: HB, P on row j = t-2 (range 1)
    {
        const int j = t - 2;
        double HB = 0.0, P = 0.0;
        if (ST || (j >= g.jA0 && j < g.jA1)) {
            HB = mm_HB(R.hb[S2(2)], R.vb[SL(1)], R.vb[SL(3)], C.ubs[S2(2) * FK_NT + g.iE],
                       C.ubs[S2(2) * FK_NT + g.iW], C.gdtcm, ctab(CT_GDTCZ, C.cj, j));
            P = -R.ha[S2(2)] * HB;
            if (!ST && j == 0 && g.ws) R.P[SL(3)] = ctab(CT_RM, C.cj, 0) * P;
        } else if (!ST && j == C.py && g.wn) P = ctab(CT_RP, C.cj, C.py - 1) * R.P[SL(3)];
        R.HB[S2(2)] = HB; R.P[SL(2)] = P;
        C.ps[S2(2) * FK_NT + i] = P;
    }
    // ---- S3: A on row j = t-3 (range 1; A_h on range 2)
    {
        const int j = t - 3;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        if (ST || (j >= g.jA0 && j < g.jA1)) {
            const double dtcz = ctab(CT_DTCZ, C.cj, j), dtf = ctab(CT_DTF, C.cj, j), dtt = ctab(CT_DTT, C.cj, j);
            if (ST || (j >= g.jH0 && j < g.jH1)) {
                const double D = mm_div(C.uas[SL(3) * FK_NT + g.iE], C.uas[SL(3) * FK_NT + g.iW], R.va[SL(2)],
                                        R.va[SL(4)], dtcz, C.dtcm, ctab(CT_RP, C.cj, j), ctab(CT_RM, C.cj, j));
                a0 = mm_Ah(R.HB[S2(3)], D);
            }
            a1 = mm_Au(R.UB[SL(3)], R.va[SL(3)], C.ps[S2(3) * FK_NT + g.iW], C.ps[S2(3) * FK_NT + g.iE], dtt, dtcz);
            a2 = mm_Av(R.vb[SL(3)], R.UB[SL(3)], R.ua[SL(3)], ctab(CT_RP, C.cj, j - 1) * R.P[SL(4)],
                       ctab(CT_RM, C.cj, j + 1) * R.P[SL(2)], dtf, dtt, C.dtcm);
            if (!ST && j == 0 && g.ws) { R.A[SL(4)][0] = a0; R.A[SL(4)][1] = a1; R.A[SL(4)][2] = -a2; }
        } else if (!ST && j == C.py && g.wn) { a0 = R.A[SL(4)][0]; a1 = R.A[SL(4)][1]; a2 = -R.A[SL(4)][2]; }
        R.A[SL(3)][0] = a0; R.A[SL(3)][1] = a1; R.A[SL(3)][2] = a2;
        double* aw = C.as + (S2(3) * 3) * FK_NT + i;
        aw[0] = a0; aw[FK_NT] = a1; aw[2 * FK_NT] = a2;
    }
    // ---- S4: lam0 on row j = t-4 (extended tile) -> in place
    {
        const int j = t - 4;
        if (ST || (j >= g.jU0 && j < g.jU1)) {
            const double dtcz = ctab(CT_DTCZ, C.cj, j);
            const double* zc_ = C.zr + (zr_slot<PH, 4>(h) * 3) * FK_NT;
            const double* zN_ = C.zr + (zr_slot<PH, 3>(h) * 3) * FK_NT + i;
            const double* zS_ = C.zr + (zr_slot<PH, 5>(h) * 3) * FK_NT + i;
            double xE[3], xW[3], xN[3], xS[3];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                xE[f] = zc_[f * FK_NT + g.iE]; xW[f] = zc_[f * FK_NT + g.iW];
                xN[f] = zN_[f * FK_NT]; xS[f] = zS_[f * FK_NT];
            }
            const double kW = C.kap - dtcz * xW[1], kE = C.kap + dtcz * xE[1];
            const double kS = C.kap - C.dtcm * xS[2], kN = C.kap + C.dtcm * xN[2];
            const double* aE = C.as + (S2(4) * 3) * FK_NT + g.iE;
            const double* aW = C.as + (S2(4) * 3) * FK_NT + g.iW;
            double out[3], su = 0.0, sv = 0.0;
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double ac = R.A[SL(4)][f];
                out[f] = ac * C.c0 + aW[f * FK_NT] * kW + aE[f * FK_NT] * kE + R.A[SL(5)][f] * kS + R.A[SL(3)][f] * kN;
                su += (xE[f] - xW[f]) * ac;
                sv += (xN[f] - xS[f]) * ac;
            }
            if (g.cU) {
                double* o = C.lcol + (j - C.gys) * C.ex;
                o[0] = out[0]; o[C.nc1] = out[1] - dtcz * su; o[2 * C.nc1] = out[2] - C.dtcm * sv;
            }
        }
    }
#undef SL
#undef S2
}

// adjoint sweep of one window (static-slot version); same contract as fk_adjoint<false>
__global__ void __launch_bounds__(FK_NT, FK_ADJ_CTAS * 128 / FK_NT) fk_adjoint2(const Sub* __restrict__ subs, const int* __restrict__ mask,
                                                        ModelP m, CostP cp, GeoP geo, const double* __restrict__ x,
                                                        const double* __restrict__ xbs,
                                                        const double* __restrict__ xfrozen,
                                                        const double* __restrict__ pred_end, const double* traj,
                                                        const double* ghost,
                                                        const long long* __restrict__ obs_start,
                                                        const int* __restrict__ obs_idx,
                                                        const double* __restrict__ obs_y,
                                                        const double* __restrict__ obs_c, double* gx, double* gw,
                                                        int nsub, double* scratch, long long slot_stride,
                                                        int* counter, const double* __restrict__ ctabp)
{
    __shared__ int s_next;
    __shared__ double zr[FK_ZR * 3 * FK_NT];
    __shared__ double uas[4 * FK_NT];
    __shared__ double ubs[2 * FK_NT];
    __shared__ double ps[2 * FK_NT];
    __shared__ double as[2 * 3 * FK_NT];
    // persistent CTA: subdomains are taken from a work counter; the adjoint variable lives in this
    // CTA's slot of an L2-persistent scratch, not in HBM
    for (;;) {
    if (threadIdx.x == 0) s_next = atomicAdd(counter, 1);
    __syncthreads();
    const int k = s_next;
    __syncthreads();
    if (k >= nsub) break;
    if (mask && !mask[k]) continue;
    const Sub s = subs[k];
    AdjCtx C;
    C.g = fk_geo(s);
    C.cj = C.g.joff + 1;
    C.tb = ctabp;
    const FkGeo& g = C.g;
    const int n3 = 3 * s.ncell;
    double* lam = scratch + (long long)blockIdx.x * slot_stride;
    C.zr = zr; C.uas = uas; C.ubs = ubs; C.ps = ps; C.as = as;
    C.nc1 = s.ncell; C.gys = s.gys; C.ex = s.ex; C.py = s.py;
    C.kap = m.kap; C.dtcm = m.dtcm; C.gdtcm = m.gdtcm; C.c0 = 1.0 - 4.0 * m.kap;
    C.lcol = lam + (g.cU ? g.li : 0);
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
    const int T = (s.py + 4 + 3) & ~3;
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
        C.col = fk_col(g, traj + s.toff + (long long)(n - 1) * n3, ghost + s.goff + (long long)(n - 1) * 3 * s.nring);
        C.tu = traj + s.toff + (long long)n * n3 + s.ncell + (g.cU ? g.li : 0);
        AdjRegs R;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            R.z[q][0] = R.z[q][1] = R.z[q][2] = 0.0; R.A[q][0] = R.A[q][1] = R.A[q][2] = 0.0;
            R.ua[q] = R.va[q] = R.vb[q] = R.UB[q] = R.P[q] = 0.0;
        }
        R.ha[0] = R.ha[1] = R.hb[0] = R.hb[1] = R.HB[0] = R.HB[1] = 0.0;
        R.l0 = R.l1 = R.l2 = R.l3 = 0.0;
        fk_load_row(g, C.col, 0, R.z[0]);
        if (g.jU0 == 0) { R.l0 = C.lcol[0]; R.l1 = C.lcol[C.nc1]; R.l2 = C.lcol[2 * C.nc1]; R.l3 = C.tu[0]; }
        // steady ticks (every stage inside its row range, no virtual rows): branch-free body
        const int ts0 = (g.jU0 + 4 + 3) & ~3, ts1 = g.jU1 - 1;
        for (int t0 = 0; t0 < T; t0 += 4) {
            const int h = t0 & 4;
            if (t0 >= ts0 && t0 + 3 <= ts1) {
                adj_tick<0, true>(t0, h, R, C); __syncthreads();
                adj_tick<1, true>(t0 + 1, h, R, C); __syncthreads();
                adj_tick<2, true>(t0 + 2, h, R, C); __syncthreads();
                adj_tick<3, true>(t0 + 3, h, R, C); __syncthreads();
            } else {
                adj_tick<0, false>(t0, h, R, C); __syncthreads();
                adj_tick<1, false>(t0 + 1, h, R, C); __syncthreads();
                adj_tick<2, false>(t0 + 2, h, R, C); __syncthreads();
                adj_tick<3, false>(t0 + 3, h, R, C); __syncthreads();
            }
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
                gg += 2.0 * (s.jw == 0 ? 1.0 : cp.bgw) * wsp * (xv - xbs[o]) * cp.ib[f];
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
    }   // persistent loop
}
