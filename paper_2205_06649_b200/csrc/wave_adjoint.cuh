// wave_adjoint.cuh -- adjoint sweep of every subdomain (step a4) and the gradient of J_ji at the window
// start, in ONE kernel; see wave_common.cuh for the design and wave_forward.cuh for the tick protocol.
//
// Warp w of the CTA runs adjoint steps m = w, w + WK_NW, ... (m-th step: lambda^n -> lambda^{n-1},
// n = W - m; eq (3)-(4) l.91-98: the window adjoint is the product of the step adjoints in reverse).
// Resident in shared memory, updated IN PLACE row by row: lambda [3][ey][ex] (zero outside the
// extended tile, so ghost cells are never stored) and u^n [ey][ex] (the step needs u^1 = u^n of the
// forward step it transposes; the warp of step m leaves u^{n-1}, which it reads anyway, for the
// warp of step m+1).  The linearisation state Z^{n-1} (trajectory store + frozen ghost ring) arrives
// through TMA bulk copies in a per-warp ring of three padded rows.
//
// The step adjoint is the transpose of Phi (model_math.cuh) about Z^{n-1}, evaluated row by row:
//   tick t:  stage A recomputed on row t-1 (h^a, u^a, v^a and the differences x_N - x_S);
//            UB, HB, P on row t-1;  A_h, A_u, A_v on row t-2;
//            L0 in SCATTER form from row t-2: A(row t-2) adds its centre and east/west parts to
//            row t-2, its southward part to row t-3 (which is then complete and stored) and
//            starts row t-1 with its northward part.  All coefficients of the scatter are local
//            to row t-2 (c_u = dtcz u0, c_v = dtcm v0), so only products cross lanes (shuffles).
// Reflective pole walls (R4): mirrored virtual rows -1 / py as in model_math.cuh; in
// scatter form the part that would leave through the wall comes back into the edge row with the
// sign of the mirrored field.
#pragma once
#include "wave_common.cuh"

template <int K> struct WaRegs {
    double z1[3][K], z2[3][K];      // Z^{n-1} rows t-1, t-2 (own columns)
    double hz2[3][2];               // E/W halo of row t-2
    double dn2[3][K];               // x_N - x_S on row t-2
    double ua2[K], va2[K], va3[K], uaL2, uaR2;
    double vb1[K], vb2[K];          // lambda_v rows t-1, t-2
    double UB2[K], HB2[K], P2[K], P3[K];
    double La[3][K], Lb[3][K];      // unfinished L0 of rows t-2 and t-3
    int pa, pe, pe2;                // row t-1 in the ring: own column 0 of field 0, the two edge-u^a cells
};
template <int K> struct WaCtx {
    WkGeo g;
    int lam, FS, u1, I_ZR, ZP, I_EW, I_EDS, I_EDE, T;
    uint32_t sm32, a_lead, a_mine, b_z, b_ew;
    unsigned gs10, need0;
    bool has_leader, have_obs, injL, injR, lane0, laneL;    // lane0 / laneL: first lane, lane 31
    int c0, lane, nchunk;
    int gcp_base, gcp_ss, gcp_rs, gcp_dst;
    unsigned tmask;
    double kap, dtcm, gdtcm, c0k, mu2;
    const double *gz, *ge, *tz;
    const WkArgs* A;
    long long qcur, qend;
    int p_pk; double p_r;
    unsigned par;                   // bits 0..2: ring slots, bits 3, 4: E/W chunk slots
};

// lane 0: padded row r of Z^{n-1} -> ring slot r % 3 (ghost rows whole, tile rows at columns 3 .. 3+ex)
template <int K>
__device__ __forceinline__ void wa_issue_row(const WaCtx<K>& C, int r, bool with_edges)
{
    const WkGeo& g = C.g;
    const int slot = r % 3;
    const uint32_t bar = C.b_z + 8u * slot;
    uint32_t dst = C.sm32 + 8u * (C.I_ZR + slot * 3 * C.ZP);
    const int lj = r - g.gys;
    const double* src; uint32_t bytes; long long fstride;
    if ((unsigned)lj < (unsigned)g.ey) { src = C.tz + lj * g.ex; bytes = g.ex * 8u; fstride = g.ncell; dst += 32u; }
    else { src = C.gz + (lj < 0 ? r : g.gys + lj - g.ey) * g.px; bytes = g.px * 8u; fstride = g.nring; }
    wk_mbar_expect32(bar, 3u * bytes + (with_edges ? (uint32_t)(g.gys + g.gyn) * 16u : 0u));
#pragma unroll 1
    for (int f = 0; f < 3; ++f) { wk_g2s32(dst, src, bytes, bar); dst += 8u * C.ZP; src += fstride; }
    if (with_edges && g.gys) wk_g2s32(C.sm32 + 8u * C.I_EDS, C.ge, g.gys * 16u, bar);
    if (with_edges && g.gyn) wk_g2s32(C.sm32 + 8u * (C.I_EDS + 8), C.ge + g.gys * 2, g.gyn * 16u, bar);
}
template <int K>
__device__ __forceinline__ void wa_issue_chunk(const WaCtx<K>& C, int c)
{
    const WkGeo& g = C.g;
    const int r0 = c * WK_EWC;
    const int rows = g.ey - r0 < WK_EWC ? g.ey - r0 : WK_EWC;
    const int slot = c & 1;
    const uint32_t bar = C.b_ew + 8u * slot;
    wk_mbar_expect32(bar, (uint32_t)rows * (3u * 48u + 16u));
    const double* src = C.gz + (g.gys + g.gyn) * g.px + r0 * 6;
    uint32_t dst = C.sm32 + 8u * (C.I_EW + slot * 18 * WK_EWC);
#pragma unroll 1
    for (int f = 0; f < 3; ++f) { wk_g2s32(dst, src, rows * 48u, bar); dst += 8u * 6 * WK_EWC; src += g.nring; }
    wk_g2s32(C.sm32 + 8u * (C.I_EDE + slot * 2 * WK_EWC), C.ge + (g.gys + g.gyn) * 2 + r0 * 2, rows * 16u, bar);
}
// row r has landed in its ring slot; for a tile row put its E/W ghost cells and edge u^a in place
template <int K>
__device__ __forceinline__ void wa_prep_row(WaCtx<K>& C, double* __restrict__ sm, int r)
{
    const WkGeo& g = C.g;
    const int slot = r % 3;
    wk_mbar_wait32(C.b_z + 8u * slot, (C.par >> slot) & 1u); C.par ^= 1u << slot;
    const int l = r - g.gys;
    if ((unsigned)l < (unsigned)g.ey) {
        const int cs = (l / WK_EWC) & 1, lr = l % WK_EWC;
        if (lr == 0) { wk_mbar_wait32(C.b_ew + 8u * cs, (C.par >> (3 + cs)) & 1u); C.par ^= 8u << cs; }
        if (C.lane < 20) sm[C.I_ZR + slot * 3 * C.ZP + C.gcp_dst] = sm[C.gcp_base + cs * C.gcp_ss + lr * C.gcp_rs];
    }
}

template <int K>
__device__ __forceinline__ void wa_tick(const int t, WaRegs<K>& R, WaCtx<K>& C, double* __restrict__ sm,
                                        const double* __restrict__ tab)
{
    const WkGeo& g = C.g;
    const int lj = t - g.gys;
    const bool tile = (unsigned)lj < (unsigned)g.ey;
    const int ci0 = C.c0 - 3;                       // tile column of own column 0
    // ---- (0) the leader has finished row t of lambda^n and u^n; H^T R^-1 (25b) forcing on that row
    if (C.has_leader) { const int nd = t + 4 < C.T + 1 ? t + 4 : C.T + 1; wk_wait_prog(C.a_lead, C.need0 + (unsigned)nd); }
    if (tile && C.have_obs) {
        const WkArgs& A = *C.A;
        for (;;) {
            const unsigned mm = __ballot_sync(0xffffffffu, (C.p_pk >> 12) == lj);
            const int cnt = __popc(mm);
            if (cnt == 0) break;
            if (C.lane < cnt) sm[C.lam + ((C.p_pk >> 8) & 3) * C.FS + lj * g.ex + (C.p_pk & 255)] += C.p_r;
            C.qcur += cnt;
            C.p_pk = 0x7fffffff;
            if (C.qcur + C.lane < C.qend) { C.p_pk = A.obs_lj[C.qcur + C.lane]; C.p_r = A.obs_r[C.qcur + C.lane]; }
            if (cnt < 32) break;
        }
        __syncwarp();
    }
    // ---- (1) loads
    const int zb = C.I_ZR + (t % 3) * 3 * C.ZP;
    int ra = 0, re = 0, re2 = 0;
    if (tile) { ra = zb + 1 + C.c0; re = zb; re2 = zb + C.ZP; }
    else if (t < g.py) { const bool north = lj >= g.ey; ra = zb + C.c0; re = C.I_EDS + (north ? 8 + (lj - g.ey) * 2 : t * 2); re2 = re + 1; }
    double z0[3][K], hz1[3][2], vb0[K], hb1[K], ub1[K], u1r[K];
    if (t < g.py) {
#pragma unroll
        for (int f = 0; f < 3; ++f)
#pragma unroll
            for (int i = 0; i < K; ++i) z0[f][i] = sm[ra + f * C.ZP + i];
    } else {
        const double sg = (t == g.py && g.wn) ? -1.0 : 1.0;     // virtual mirrored row py
#pragma unroll
        for (int i = 0; i < K; ++i) { z0[0][i] = R.z1[0][i]; z0[1][i] = R.z1[1][i]; z0[2][i] = sg * R.z1[2][i]; }
    }
#pragma unroll
    for (int f = 0; f < 3; ++f) { hz1[f][0] = sm[R.pa + f * C.ZP - 1]; hz1[f][1] = sm[R.pa + f * C.ZP + K]; }
    const double eL = sm[R.pe], eR = sm[R.pe2];
    {
        const int o0 = C.lam + lj * g.ex + ci0;     // lambda row t (v), row t-1 (h, u), u^n row t-1
        const bool tile1 = (unsigned)(lj - 1) < (unsigned)g.ey;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const bool tc = (C.tmask >> i) & 1u;
            vb0[i] = (tile && tc) ? sm[o0 + 2 * C.FS + i] : 0.0;
            hb1[i] = (tile1 && tc) ? sm[o0 - g.ex + i] : 0.0;
            ub1[i] = (tile1 && tc) ? sm[o0 - g.ex + C.FS + i] : 0.0;
            u1r[i] = (tile1 && tc) ? sm[C.u1 + (lj - 1) * g.ex + ci0 + i] : 0.0;
        }
    }
    if (g.wn && t == g.py) {                        // virtual row py: lambda_v mirrored
#pragma unroll
        for (int i = 0; i < K; ++i) vb0[i] = -R.vb1[i];
    }
    if (g.ws && t <= 2) {                           // virtual row -1
        if (t == 1) {
#pragma unroll
            for (int i = 0; i < K; ++i) { R.z2[0][i] = R.z1[0][i]; R.z2[1][i] = R.z1[1][i]; R.z2[2][i] = -R.z1[2][i]; R.vb2[i] = -R.vb1[i]; }
        }
        if (t == 2) {
            const double rm0 = tab[8 + WK_T_RM];
#pragma unroll
            for (int i = 0; i < K; ++i) { R.va3[i] = -R.va2[i]; R.P3[i] = rm0 * R.P2[i]; }
        }
    }

    // ---- (2) row t-1: stage A recomputed, UB, HB, P
    double ua1[K], va1[K], dn1[3][K], UB1[K], HB1[K], P1[K], uaL1, uaR1;
    if (t <= g.py) {
        const double* tb = tab + t * 8;
        const double dtcz1 = tb[WK_T_DTCZ], gdtcz1 = tb[WK_T_GDTCZ], dtf1 = tb[WK_T_DTF], dtt1 = tb[WK_T_DTT];
        double ha1[K];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double cu = dtcz1 * R.z1[1][i], cv = C.dtcm * R.z1[2][i];
            double xa[3];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double xE = i < K - 1 ? R.z1[f][i + 1 < K ? i + 1 : i] : hz1[f][1];
                const double xW = i > 0 ? R.z1[f][i > 0 ? i - 1 : 0] : hz1[f][0];
                dn1[f][i] = z0[f][i] - R.z2[f][i];
                xa[f] = R.z1[f][i] - (cu * (xE - xW) + cv * dn1[f][i]) +
                        C.kap * (xE + xW + z0[f][i] + R.z2[f][i] - 4.0 * R.z1[f][i]);
            }
            ha1[i] = xa[0]; ua1[i] = xa[1]; va1[i] = xa[2];
            UB1[i] = mm_UB(ub1[i], R.vb1[i], u1r[i], dtf1, dtt1);
        }
        uaL1 = wk_up(ua1[K - 1]); uaR1 = wk_dn(ua1[0]);
        uaL1 = C.injL ? eL : uaL1; uaR1 = C.injR ? eR : uaR1;
        double UBL = wk_up(UB1[K - 1]), UBR = wk_dn(UB1[0]);
        UBL = C.lane0 ? 0.0 : UBL; UBR = C.laneL ? 0.0 : UBR;      // ghost columns: lambda = 0
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double UE = i < K - 1 ? UB1[i + 1 < K ? i + 1 : i] : UBR;
            const double UW = i > 0 ? UB1[i > 0 ? i - 1 : 0] : UBL;
            HB1[i] = mm_HB(hb1[i], vb0[i], R.vb2[i], UE, UW, C.gdtcm, gdtcz1);
            P1[i] = -ha1[i] * HB1[i];
        }
    } else {
        const bool vr = g.wn && t == g.py + 1;      // virtual row py: v^a mirrored, P carries the metric ratio
        const double rpn = tab[g.py * 8 + WK_T_RP];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            ua1[i] = 0.0; va1[i] = vr ? -R.va2[i] : 0.0; UB1[i] = 0.0; HB1[i] = 0.0; P1[i] = vr ? rpn * R.P2[i] : 0.0;
#pragma unroll
            for (int f = 0; f < 3; ++f) dn1[f][i] = 0.0;
        }
        uaL1 = 0.0; uaR1 = 0.0;
    }

    // ---- (3) row t-2: A_h, A_u, A_v; (4) scatter into L0 of rows t-1, t-2, t-3
    double Lc[3][K];
    if (t >= 2 && t <= g.py + 1) {               // (rows -1 and py are virtual: nothing is scattered from them)
        const double* tb = tab + t * 8 - 8;
        const double dtcz2 = tb[WK_T_DTCZ], dtf2 = tb[WK_T_DTF], dtt2 = tb[WK_T_DTT], rp2 = tb[WK_T_RP], rm2 = tb[WK_T_RM];
        const double rp3 = tb[WK_T_RP - 8], rm1 = tb[WK_T_RM + 8];
        double PL = wk_up(R.P2[K - 1]), PR = wk_dn(R.P2[0]);
        PL = C.lane0 ? 0.0 : PL; PR = C.laneL ? 0.0 : PR;
        double Aa[3][K], mE[3][K], mW[3][K];
        const bool wallS = g.ws && t == 2, wallN = g.wn && t == g.py + 1;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double uE = i < K - 1 ? R.ua2[i + 1 < K ? i + 1 : i] : R.uaR2;
            const double uW = i > 0 ? R.ua2[i > 0 ? i - 1 : 0] : R.uaL2;
            const double PE = i < K - 1 ? R.P2[i + 1 < K ? i + 1 : i] : PR;
            const double PW = i > 0 ? R.P2[i > 0 ? i - 1 : 0] : PL;
            const double D = mm_div(uE, uW, va1[i], R.va3[i], dtcz2, C.dtcm, rp2, rm2);
            Aa[0][i] = mm_Ah(R.HB2[i], D);
            Aa[1][i] = mm_Au(R.UB2[i], R.va2[i], PW, PE, dtt2, dtcz2);
            Aa[2][i] = mm_Av(R.vb2[i], R.UB2[i], R.ua2[i], rp3 * R.P3[i], rm1 * P1[i], dtf2, dtt2, C.dtcm);
            const double cu = dtcz2 * R.z2[1][i], cv = C.dtcm * R.z2[2][i];
            const double kE = C.kap - cu, kW = C.kap + cu, kS = C.kap + cv, kN = C.kap - cv;
            double su = 0.0, sv = 0.0;
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double a = Aa[f][i];
                const double xE = i < K - 1 ? R.z2[f][i + 1 < K ? i + 1 : i] : R.hz2[f][1];
                const double xW = i > 0 ? R.z2[f][i > 0 ? i - 1 : 0] : R.hz2[f][0];
                mE[f][i] = a * kE; mW[f][i] = a * kW;
                su += (xE - xW) * a; sv += R.dn2[f][i] * a;
                const double sgn = f == 2 ? -1.0 : 1.0;
                const double mS = a * kS, mN = a * kN;
                double la = R.La[f][i] + a * C.c0k;
                if (wallS) la += sgn * mS; else R.Lb[f][i] += mS;
                if (wallN) { la += sgn * mN; Lc[f][i] = 0.0; } else Lc[f][i] = mN;
                R.La[f][i] = la;
            }
            R.La[1][i] -= dtcz2 * su; R.La[2][i] -= C.dtcm * sv;
        }
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            const double fW = wk_up(mE[f][K - 1]), fE = wk_dn(mW[f][0]);
#pragma unroll
            for (int i = 0; i < K; ++i)
                R.La[f][i] += (i > 0 ? mE[f][i > 0 ? i - 1 : 0] : fW) + (i < K - 1 ? mW[f][i + 1 < K ? i + 1 : i] : fE);
        }
    } else {
#pragma unroll
        for (int f = 0; f < 3; ++f)
#pragma unroll
            for (int i = 0; i < K; ++i) Lc[f][i] = 0.0;
    }

    // ---- (5) row t-3 of lambda^{n-1} is complete; u^{n-1} of row t-2 replaces u^n
    {
        const int l3 = lj - 3, l2 = lj - 2;
        if ((unsigned)l3 < (unsigned)g.ey) {
            const int o3 = C.lam + l3 * g.ex + ci0;
#pragma unroll
            for (int i = 0; i < K; ++i)
                if ((C.tmask >> i) & 1u) { sm[o3 + i] = R.Lb[0][i]; sm[o3 + C.FS + i] = R.Lb[1][i]; sm[o3 + 2 * C.FS + i] = R.Lb[2][i]; }
        }
        if ((unsigned)l2 < (unsigned)g.ey) {
            const int o2 = C.u1 + l2 * g.ex + ci0;
#pragma unroll
            for (int i = 0; i < K; ++i)
                if ((C.tmask >> i) & 1u) sm[o2 + i] = R.z2[1][i];
        }
    }
    // the next row of Z^{n-1} must have landed; its ghost cells go in place
    if (t + 1 < g.py) wa_prep_row<K>(C, sm, t + 1);
    __syncwarp();
    // ---- (6) one lane: progress word, the row after next, next E/W chunk
    if (wk_elect()) {
        if (t < C.T) wk_publish(C.a_mine, C.gs10 + (unsigned)t + 1u);
        if (t + 2 < g.py) wa_issue_row<K>(C, t + 2, false);
        const int l1 = lj + 1;
        if ((unsigned)l1 < (unsigned)g.ey && (l1 % WK_EWC) == WK_EWC - 1 && l1 / WK_EWC + 2 < C.nchunk)
            wa_issue_chunk<K>(C, l1 / WK_EWC + 2);
    }
    // ---- (7) rotate
#pragma unroll
    for (int i = 0; i < K; ++i) {
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            R.z2[f][i] = R.z1[f][i]; R.z1[f][i] = z0[f][i]; R.dn2[f][i] = dn1[f][i];
            R.Lb[f][i] = R.La[f][i]; R.La[f][i] = Lc[f][i];
        }
        R.ua2[i] = ua1[i]; R.va3[i] = R.va2[i]; R.va2[i] = va1[i];
        R.vb2[i] = R.vb1[i]; R.vb1[i] = vb0[i];
        R.UB2[i] = UB1[i]; R.HB2[i] = HB1[i]; R.P3[i] = R.P2[i]; R.P2[i] = P1[i];
    }
#pragma unroll
    for (int f = 0; f < 3; ++f) { R.hz2[f][0] = hz1[f][0]; R.hz2[f][1] = hz1[f][1]; }
    R.uaL2 = uaL1; R.uaR2 = uaR1;
    if (t < g.py) { R.pa = ra; R.pe = re; R.pe2 = re2; }
}

template <int K>
__global__ void __launch_bounds__(WK_NT, 1) wk_adjoint(const __grid_constant__ WkArgs A)
{
    extern __shared__ __align__(128) double sm[];
    const int tid = threadIdx.x, lane = tid & 31, w = wk_uni(tid >> 5);
    const WkLayout Ly = wk_layout(true, A.maxex, A.maxey, A.maxpx, A.maxpy);
    const uint32_t sm32 = wk_s32(sm);
    int* s_next = reinterpret_cast<int*>(sm + 52);
    double* tab = sm + Ly.tab;
    const int IW = Ly.wbase + w * Ly.wsz;
    if (tid == 0) {
        for (int i = 0; i < 41; ++i) wk_mbar_init32(sm32 + 8u * i, 1);
        wk_fence_mbar_init();
    }
    if (tid < WK_NW) reinterpret_cast<unsigned*>(sm + 48)[tid] = 0u;
    for (int q = tid; q < Ly.total - WK_HDR; q += WK_NT) sm[WK_HDR + q] = 0.0;
    __syncthreads();
    unsigned gbase = 1u;
    const int lw = (w + WK_NW - 1) % WK_NW;

    WaCtx<K> C;
    C.lam = Ly.st; C.u1 = Ly.u1; C.ZP = Ly.ZP;
    C.I_ZR = IW + Ly.zr; C.I_EW = IW + Ly.ew; C.I_EDS = IW + Ly.eds; C.I_EDE = IW + Ly.ede;
    C.sm32 = sm32; C.a_lead = sm32 + 8u * 48u + 4u * lw; C.a_mine = sm32 + 8u * 48u + 4u * w;
    C.b_z = sm32 + 8u * (w * 5); C.b_ew = sm32 + 8u * (w * 5 + 3);
    C.c0 = 2 + K * lane; C.lane = lane; C.lane0 = lane == 0; C.laneL = lane == 31;
    C.kap = A.m.kap; C.dtcm = A.m.dtcm; C.gdtcm = A.m.gdtcm; C.c0k = 1.0 - 4.0 * A.m.kap; C.mu2 = 2.0 * A.cp.mu;
    C.A = &A; C.par = 0u;
    const int lam = Ly.st;

    for (;;) {
        if (tid == 0) *s_next = atomicAdd(A.counter, 1);
        __syncthreads();
        const int k = wk_uni(*s_next);
        __syncthreads();
        if (k >= A.nsub) break;
        if (A.mask && !A.mask[k]) continue;
        const Sub s = A.subs[k];
        const WkGeo g = wk_geo(s);
        C.g = g;
        const int FS = g.ncell;                 // lambda and u^n are stored with the tile's own pitch
        C.FS = FS;
        const long long n3 = 3LL * g.ncell;

        // ---------------- init: lambda^W = successor-window overlap forcing (25c), else zero; u^W
        wk_load_tab(tab, A.m, g);
        {
            const bool succ = s.jw < A.geo.q - 1;
            const double* tw = A.traj + s.toff + (long long)g.W * n3;
            const double* xn = succ ? A.xfrozen + A.subs[k + A.geo.p1 * A.geo.p2].coff : nullptr;
            for (int c = tid; c < g.ncell; c += WK_NT) {
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    const double zv = __ldg(tw + (long long)f * g.ncell + c);
                    sm[lam + f * FS + c] = succ ? C.mu2 * (zv - __ldg(xn + (long long)f * g.ncell + c)) * A.cp.ib[f] : 0.0;
                    if (f == 1) sm[C.u1 + c] = zv;
                }
            }
        }
        __syncthreads();

        // ---------------- per-lane column map of this tile
        C.tmask = 0u;
#pragma unroll
        for (int i = 0; i < K; ++i) if ((C.c0 + i >= 3) && (C.c0 + i < 3 + g.ex)) C.tmask |= 1u << i;
        C.injL = lane == 0; C.injR = (lane == 31) && (C.c0 + K == g.px - 2);
        if (lane < 18) {                        // E/W ghost cell (field lane/6, cell lane%6) -> padded columns 0..2, px-3..px-1
            const int f = lane / 6, e = lane % 6;
            C.gcp_base = C.I_EW + f * 6 * WK_EWC + e; C.gcp_ss = 18 * WK_EWC; C.gcp_rs = 6;
            C.gcp_dst = f * C.ZP + 1 + (e < 3 ? e : g.ex + e);
        } else {                                // lanes 18, 19: edge u^a west / east -> the free cell 0 of fields 0 / 1
            C.gcp_base = C.I_EDE + (lane - 18); C.gcp_ss = 2 * WK_EWC; C.gcp_rs = 2;
            C.gcp_dst = (lane - 18) * C.ZP;
        }
        C.nchunk = (g.ey + WK_EWC - 1) / WK_EWC;
        C.T = g.py + 3;

        // ---------------- the steps of this warp
        for (int m = w; m < g.W; m += WK_NW) {
            const int n = g.W - m;
            const unsigned gs = gbase + (unsigned)m;
            C.gs10 = gs << 10; C.need0 = (gs - 1u) << 10; C.has_leader = m > 0;
            C.gz = A.ghost + s.goff + (long long)(n - 1) * 3 * g.nring;
            C.ge = A.gedge + s.eoff + (long long)(n - 1) * 2 * g.py;
            C.tz = A.traj + s.toff + (long long)(n - 1) * n3;
            C.qcur = 0; C.qend = 0;
            if (A.obs_start) { C.qcur = A.obs_start[s.ooff + n]; C.qend = A.obs_start[s.ooff + n + 1]; }
            C.have_obs = C.qend > C.qcur;
            C.p_pk = 0x7fffffff; C.p_r = 0.0;
            if (C.have_obs && C.qcur + lane < C.qend) { C.p_pk = A.obs_lj[C.qcur + lane]; C.p_r = A.obs_r[C.qcur + lane]; }
            if (wk_elect()) {
                wa_issue_row<K>(C, 0, true);
                if (g.py > 1) wa_issue_row<K>(C, 1, false);
                wa_issue_chunk<K>(C, 0);
                if (C.nchunk > 1) wa_issue_chunk<K>(C, 1);
            }
            WaRegs<K> R;
#pragma unroll
            for (int i = 0; i < K; ++i) {
#pragma unroll
                for (int f = 0; f < 3; ++f) { R.z1[f][i] = R.z2[f][i] = R.dn2[f][i] = R.La[f][i] = R.Lb[f][i] = 0.0; }
                R.ua2[i] = R.va2[i] = R.va3[i] = R.vb1[i] = R.vb2[i] = R.UB2[i] = R.HB2[i] = R.P2[i] = R.P3[i] = 0.0;
            }
#pragma unroll
            for (int f = 0; f < 3; ++f) { R.hz2[f][0] = 0.0; R.hz2[f][1] = 0.0; }
            R.uaL2 = R.uaR2 = 0.0; R.pa = C.I_ZR + 1; R.pe = C.I_EDS; R.pe2 = C.I_EDS;
            wa_prep_row<K>(C, sm, 0);           // (the ring is private to this warp: no leader involved)
            __syncwarp();
#pragma unroll 1
            for (int t = 0; t < C.T; ++t) wa_tick<K>(t, R, C, sm, tab);
            if (wk_elect()) wk_publish(C.a_mine, C.gs10 + (unsigned)C.T + 1u);
            __syncwarp();
        }
        __syncthreads();

        // ---------------- gradient at the window start: lambda^0 + H^T R^-1 at level 0 (25b)
        //                  + (25a) + control-level (25c) terms; g_w = sigma_b g_x (eq (44) l.630-634)
        if (A.obs_start) {
            const long long a0 = A.obs_start[s.ooff], a1 = A.obs_start[s.ooff + 1];
            for (long long q = a0 + tid; q < a1; q += WK_NT) {
                const int pk = A.obs_lj[q];
                sm[lam + ((pk >> 8) & 3) * FS + (pk >> 12) * g.ex + (pk & 255)] += A.obs_r[q];
            }
            __syncthreads();
        }
        {
            const bool pred = s.jw > 0;
            for (int lj = w; lj < g.ey; lj += WK_NW) {
                const int nr = A.geo.nrowcov[s.ej0 + lj];
                for (int li = lane; li < g.ex; li += 32) {
                    int gi = s.ei0 + li; gi = gi < 0 ? gi + A.geo.nlon : (gi >= A.geo.nlon ? gi - A.geo.nlon : gi);
                    const double wsp2 = 2.0 * (s.jw == 0 ? 1.0 : A.cp.bgw) / (double)(A.geo.ncolcov[gi] * nr);
                    const int c = lj * g.ex + li;
#pragma unroll
                    for (int f = 0; f < 3; ++f) {
                        const long long o = s.coff + (long long)f * g.ncell + c;
                        const double xv = __ldg(A.x + o);
                        double gg = sm[lam + f * FS + c] + wsp2 * (xv - __ldg(A.xbs + o)) * A.cp.ib[f];
                        if (pred) gg += C.mu2 * (xv - __ldg(A.pred_end + o)) * A.cp.ib[f];
                        sm[lam + f * FS + c] = gg;
                    }
                }
            }
            for (int r = 0; r < s.nnb; ++r) {   // (25c) case 1, one rectangle at a time (a cell may lie in several)
                __syncthreads();
                const NbRect nb = A.nbr[s.nb0 + r];
                const double* xf = A.xfrozen + nb.coff2 + (long long)nb.nj0 * nb.ex2 + nb.ni0;
                for (int dj = w; dj < nb.h; dj += WK_NW)
                    for (int di = lane; di < nb.w; di += 32) {
                        const int c = (nb.j0 + dj) * g.ex + nb.i0 + di;
#pragma unroll
                        for (int f = 0; f < 3; ++f) {
                            const double xv = __ldg(A.x + s.coff + (long long)f * g.ncell + c);
                            sm[lam + f * FS + c] += C.mu2 * (xv - __ldg(xf + (long long)f * nb.ncell2 + dj * nb.ex2 + di)) * A.cp.ib[f];
                        }
                    }
            }
            __syncthreads();
            for (int c = tid; c < g.ncell; c += WK_NT) {
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    const long long o = s.coff + (long long)f * g.ncell + c;
                    const double gg = sm[lam + f * FS + c];
                    A.gx[o] = gg;
                    if (A.gw) A.gw[o] = A.cp.sb[f] * gg;
                }
            }
        }
        gbase += (unsigned)g.W + 1u;
    }
}
