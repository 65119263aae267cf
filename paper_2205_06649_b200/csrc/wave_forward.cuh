// wave_forward.cuh -- forward sweep of every subdomain (step a1), trajectory store (a2) and the cost
// terms of J_ji (a3, eq (25) l.338-344) in ONE kernel; see wave_common.cuh for the design.
//
// Warp w of the CTA runs model steps n = w, w + WK_NW, ... of the window.  Its input level Z^n is
// the resident state in shared memory, which the warp of step n-1 (the leader) is still writing
// a few rows ahead; its output Z^{n+1} overwrites the same rows in place three rows behind its
// own read position and leaves for the trajectory store as TMA bulk stores, one per tile row and
// field.  One tick t of a warp:
//     read padded row t (own K columns) and the E/W halo of row t-1
//     stage A   on row t-1  (advection + diffusion, eq (60)-(62) advective part, R3)
//     h^1, u^1  on row t-2  (forward-backward gravity / Coriolis step)
//     v^1       on row t-3  -> row t-3 of Z^{n+1} is complete: shared memory, TMA store, H (25b)
// East/west neighbours inside a lane's K columns are registers, across lanes one shuffle; the
// value of u^a in the ghost columns 1 and px-2 (needed by h^1 in columns 2 and px-3, not owned by
// any lane when px - 4 = 32 K) is frozen boundary data precomputed by xk_edge_ua.
// Synchronisation: after tick t a warp publishes (step << 10) + t + 1; the warp of the next step
// starts its tick t when its leader has published tick t + 3 (row t of its input is then final,
// and the leader's bulk store of every row this warp is about to overwrite has left shared memory).
// The first step of a subdomain (n = 0) follows the LAST step of the previous subdomain of this CTA: its
// input rows, the control, arrive from global memory two ticks ahead (TMA into the resident rows the
// previous subdomain has finished with); all cost terms of J_ji (the misfits H Z^n - y included, sampled from the
// trajectory store: 2 % of the points), the level-0 copy of the trajectory store and the successor-window term
// run in ck_cost (cost_kernels.cuh) after this kernel: with observations every 8th level and 8 steps in flight
// one of the steps of the pipeline always carried observations and set the pace of all (7 % of the kernel).
// The ticks without a wall event run a steady body, one tick per loop iteration (the hot loop must stay inside the
// instruction cache: unrolling by 3 or 6 was slower, profiles/r2_wave_v2.md); the others a general body with uniform branches.
#pragma once
#include "wave_common.cuh"

#define WK_XD 3         // a first step fetches its control rows this many ticks ahead (4 mbarrier slots: WK_XD <= 3)


// row histories of one warp-step (names: 1 = row t-1, 2 = row t-2, ... at the start of tick t)
template <int K> struct WfRegs {
    double z1[3][K], z2[3][K], ha2[K], ua2[K], va2[K], va3[K], h13[K], h14[K], u13[K];
    double uaL2, uaR2;
    int pa, pfs, pe;                // row t-1: own column 0 of field 0 at sm[pa], field stride, edge-u^a index
};
// everything a tick needs besides the histories (uniform unless noted)
template <int K> struct WfCtx {
    WkGeo g;
    static constexpr int P = WK_AZP(K), FS = WK_AROWS(K) * WK_AZP(K);     // row pitch, field stride (compile-time, wave_common.cuh)
    int st, I_SN, I_EW, I_EDS, I_EDE, T;
    uint32_t sm32, a_lead, a_mine, b_sn, b_ew;      // shared-window addresses: progress words, barriers
    unsigned gs10, need0;                            // (global step << 10), ((global step - 1) << 10)
    bool has_leader, injL, injR;                     // injL / injR per lane
    bool first;                                      // step 0 of a subdomain: its input rows (the control) arrive from global memory
    int dlead, TLd;                                  // tick t starts when the leader has published min(t + dlead, TLd + 1)
    uint32_t b_x;                                    // mbarriers of the control rows in flight (4 slots)
    const double* xk;                                // control of this subdomain [3][ey][ex]
    int c0, lane, nchunk;
    int gcp_base, gcp_ss, gcp_rs, gcp_dst;           // per lane (< 20): ghost / edge cell copied per tile row
    unsigned tmask;                                  // per lane: bit i = own column i is a tile column
    double kap, dtcm, gdtcm;
    const double *gz, *ge; double* tout;
    const WkArgs* A;
    unsigned par;
};
template <int K>
__device__ __forceinline__ void wf_issue_chunk(const WfCtx<K>& C, int c)
{   // lane 0: E/W ghost cells + edge u^a of tile rows [c*EWC, ...) -> staging slot c & 1
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
template <int K>
__device__ __forceinline__ void wf_issue_ns(const WfCtx<K>& C, bool north)
{   // lane 0: the three ghost rows of one side + their edge u^a
    const WkGeo& g = C.g;
    const int rows = north ? g.gyn : g.gys;
    const int roff = north ? g.gys : 0;
    wk_mbar_expect32(C.b_sn, (uint32_t)rows * (3u * g.px * 8u + 16u));
    const double* src = C.gz + roff * g.px;
    uint32_t dst = C.sm32 + 8u * C.I_SN;
#pragma unroll 1
    for (int f = 0; f < 3; ++f) { wk_g2s32(dst, src, rows * g.px * 8u, C.b_sn); dst += 8u * 3 * g.px; src += g.nring; }
    wk_g2s32(C.sm32 + 8u * (C.I_EDS + (north ? 8 : 0)), C.ge + roff * 2, rows * 16u, C.b_sn);
}

// lane 0, first step of a subdomain: tile row l of the control -> resident state (slot l & 3)
template <int K>
__device__ __forceinline__ void wf_issue_xrow(const WfCtx<K>& C, int l)
{
    const WkGeo& g = C.g;
    const uint32_t bar = C.b_x + 8u * (l & 3);
    wk_mbar_expect32(bar, 3u * g.ex * 8u);
    const double* src = C.xk + l * g.ex;
    uint32_t dst = C.sm32 + 8u * (C.st + l * C.P);
#pragma unroll 1
    for (int f = 0; f < 3; ++f) { wk_g2s32(dst, src, g.ex * 8u, bar); dst += 8u * C.FS; src += g.ncell; }
}
template <int K>
__device__ __forceinline__ void wf_wait_xrow(WfCtx<K>& C, int l)
{
    const int slot = l & 3;
    wk_mbar_wait32(C.b_x + 8u * slot, (C.par >> (4 + slot)) & 1u); C.par ^= 16u << slot;
}

// put the E/W ghost cells (lanes 0..17) and the edge u^a (lanes 18, 19) of tile row l next to the row
template <int K>
__device__ __forceinline__ void wf_prep_row(WfCtx<K>& C, double* __restrict__ sm, int l)
{
    const int slot = (l / WK_EWC) & 1, lr = l % WK_EWC;
    if (lr == 0) { wk_mbar_wait32(C.b_ew + 8u * slot, (C.par >> (1 + slot)) & 1u); C.par ^= 2u << slot; }
    if (C.lane < 20) sm[C.st + l * C.P + C.gcp_dst] = sm[C.gcp_base + slot * C.gcp_ss + lr * C.gcp_rs];
}

template <int K>
__device__ __forceinline__ void wf_tick(const int t, WfRegs<K>& R, WfCtx<K>& C, double* __restrict__ sm,
                                        const double* __restrict__ tab)
{
    const WkGeo& g = C.g;
    const int lj = t - g.gys;                       // tile row of padded row t (if it is one)
    const bool tile = (unsigned)lj < (unsigned)g.ey;
    // ---- (0) row t becomes readable
    if (C.has_leader && !(t & 1)) {             // (one poll for two ticks: every even tick waits for what the next one needs)
        const int nd = t + 1 + C.dlead < C.TLd + 1 ? t + 1 + C.dlead : C.TLd + 1; wk_wait_prog(C.a_lead, C.need0 + (unsigned)nd);
    }
    int ra = 0, rfs = 0, re = 0;                    // own column 0 of row t, field stride, edge-u^a index
    if (tile) {                                      // (its E/W ghost cells were put in place one tick earlier)
        if (C.first) wf_wait_xrow<K>(C, lj);
        const int rowb = C.st + lj * C.P;
        ra = rowb - 3 + C.c0; rfs = C.FS; re = rowb + g.ex + 3;
    } else if (t < g.py) {
        const bool north = lj >= g.ey;
        if (t == 0 || lj == g.ey) { wk_mbar_wait32(C.b_sn, C.par & 1u); C.par ^= 1u; }
        const int rr = north ? lj - g.ey : t;
        ra = C.I_SN + rr * g.px + C.c0; rfs = 3 * g.px; re = C.I_EDS + (north ? 8 : 0) + rr * 2;
    }
    // ---- (1) loads: own columns of row t, E/W halo of row t-1
    double z0[3][K], hz[3][2];
    if (t < g.py) {
#pragma unroll
        for (int f = 0; f < 3; ++f)
#pragma unroll
            for (int i = 0; i < K; ++i) z0[f][i] = sm[ra + f * rfs + i];
    } else {
        const double sg = (t == g.py && g.wn) ? -1.0 : 1.0;     // virtual mirrored row py
#pragma unroll
        for (int i = 0; i < K; ++i) { z0[0][i] = R.z1[0][i]; z0[1][i] = R.z1[1][i]; z0[2][i] = sg * R.z1[2][i]; }
    }
#pragma unroll
    for (int f = 0; f < 3; ++f) { hz[f][0] = sm[R.pa + f * R.pfs - 1]; hz[f][1] = sm[R.pa + f * R.pfs + K]; }
    const double eL = sm[R.pe], eR = sm[R.pe + 1];
    if (g.ws && t <= 3) {                            // virtual mirrored row -1 (R4)
        if (t == 1) {
#pragma unroll
            for (int i = 0; i < K; ++i) { R.z2[0][i] = R.z1[0][i]; R.z2[1][i] = R.z1[1][i]; R.z2[2][i] = -R.z1[2][i]; }
        }
        if (t == 2) {
#pragma unroll
            for (int i = 0; i < K; ++i) R.va3[i] = -R.va2[i];
        }
        if (t == 3) {
#pragma unroll
            for (int i = 0; i < K; ++i) R.h14[i] = R.h13[i];
        }
    }

    // ---- (2) stage A on row t-1 (garbage, never used, at t = 0)
    double ha1[K], ua1[K], va1[K], uaL1, uaR1;
    if (t <= g.py) {
        const double dtcz1 = tab[t * 8 + WK_T_DTCZ];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double cu = dtcz1 * R.z1[1][i], cv = C.dtcm * R.z1[2][i];
            double xa[3];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double xE = i < K - 1 ? R.z1[f][i + 1 < K ? i + 1 : i] : hz[f][1];
                const double xW = i > 0 ? R.z1[f][i > 0 ? i - 1 : 0] : hz[f][0];
                xa[f] = mm_stageA(R.z1[f][i], xE, xW, z0[f][i], R.z2[f][i], cu, cv, C.kap);
            }
            ha1[i] = xa[0]; ua1[i] = xa[1]; va1[i] = xa[2];
        }
        uaL1 = wk_up(ua1[K - 1]); uaR1 = wk_dn(ua1[0]);
        uaL1 = C.injL ? eL : uaL1;                   // frozen u^a of the ghost columns 1 and px-2 (xk_edge_ua)
        uaR1 = C.injR ? eR : uaR1;
    } else {
        const double sg = (t == g.py + 1 && g.wn) ? -1.0 : 0.0;  // virtual row py: v^a mirrored
#pragma unroll
        for (int i = 0; i < K; ++i) { ha1[i] = 0.0; ua1[i] = 0.0; va1[i] = sg * R.va2[i]; }
        uaL1 = 0.0; uaR1 = 0.0;
    }

    // ---- (3) h^1 and u^1 on row t-2
    double h12[K], u12[K];
    if (t <= g.py + 1) {
        const double* tb = tab + t * 8 - 8;
        const double dtcz2 = tb[WK_T_DTCZ], gdtcz2 = tb[WK_T_GDTCZ], dtf2 = tb[WK_T_DTF], dtt2 = tb[WK_T_DTT];
        const double rp2 = tb[WK_T_RP], rm2 = tb[WK_T_RM];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double uE = i < K - 1 ? R.ua2[i + 1 < K ? i + 1 : i] : R.uaR2;
            const double uW = i > 0 ? R.ua2[i > 0 ? i - 1 : 0] : R.uaL2;
            h12[i] = mm_h1(R.ha2[i], mm_div(uE, uW, va1[i], R.va3[i], dtcz2, C.dtcm, rp2, rm2));
        }
        const double hL = wk_up(h12[K - 1]), hR = wk_dn(h12[0]);
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double hE = i < K - 1 ? h12[i + 1 < K ? i + 1 : i] : hR;
            const double hW = i > 0 ? h12[i > 0 ? i - 1 : 0] : hL;
            u12[i] = mm_u1(R.ua2[i], R.va2[i], hE, hW, gdtcz2, dtf2, dtt2);
        }
    } else {
#pragma unroll
        for (int i = 0; i < K; ++i) { h12[i] = (t == g.py + 2 && g.wn) ? R.h13[i] : 0.0; u12[i] = 0.0; }
    }
    // ---- (4) v^1 on row t-3: row t-3 of Z^{n+1} is complete
    const int l3 = lj - 3;
    const bool out = (unsigned)l3 < (unsigned)g.ey;
    if (out) {
        const double dtf3 = tab[t * 8 - 16 + WK_T_DTF], dtt3 = tab[t * 8 - 16 + WK_T_DTT];
        const int ob0 = C.st + l3 * C.P + C.c0 - 3;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double v1 = mm_v1(R.va3[i], R.u13[i], h12[i], R.h14[i], C.gdtcm, dtf3, dtt3);
            if ((C.tmask >> i) & 1u) { sm[ob0 + i] = R.h13[i]; sm[ob0 + C.FS + i] = R.u13[i]; sm[ob0 + 2 * C.FS + i] = v1; }
        }
    }
    wk_fence_async();
    // E/W ghost cells and edge u^a of the NEXT row go next to its tile row (the leader read them two ticks ago)
    const int l1 = lj + 1;
    const bool prep = (unsigned)l1 < (unsigned)g.ey;
    if (prep) wf_prep_row<K>(C, sm, l1);
    __syncwarp();
    // ---- (5) one lane: progress word, trajectory stores, refills of the staging buffers
    if (wk_elect()) {
        // a follower overwrites row r after my tick r+6 is published: the store issued three ticks ago must have left
        if (out) wk_wait_read<2>(); else wk_wait_read<0>();
        if (t < C.T) wk_publish(C.a_mine, C.gs10 + (unsigned)t + 1u);
        if (out) {
            uint32_t src = C.sm32 + 8u * (C.st + l3 * C.P);
            double* dst = C.tout + l3 * g.ex;
#pragma unroll 1
            for (int f = 0; f < 3; ++f) { wk_s2g32(dst, src, g.ex * 8u); dst += g.ncell; src += 8u * C.FS; }
            wk_commit();
        }
        if (g.gys && g.gyn && t == g.gys) wf_issue_ns(C, true);               // S rows consumed (halo of row gys-1 read)
        if (C.first && (unsigned)(lj + WK_XD) < (unsigned)g.ey) wf_issue_xrow<K>(C, lj + WK_XD);
        if (prep && (l1 % WK_EWC) == WK_EWC - 1 && l1 / WK_EWC + 2 < C.nchunk) wf_issue_chunk(C, l1 / WK_EWC + 2);
    }
    // ---- (6) rotate the row histories
#pragma unroll
    for (int i = 0; i < K; ++i) {
#pragma unroll
        for (int f = 0; f < 3; ++f) { R.z2[f][i] = R.z1[f][i]; R.z1[f][i] = z0[f][i]; }
        R.ha2[i] = ha1[i]; R.ua2[i] = ua1[i]; R.va3[i] = R.va2[i]; R.va2[i] = va1[i];
        R.h14[i] = R.h13[i]; R.h13[i] = h12[i]; R.u13[i] = u12[i];
    }
    R.uaL2 = uaL1; R.uaR2 = uaR1;
    if (t < g.py) { R.pa = ra; R.pfs = rfs; R.pe = re; }
}

// The same tick for the rows well inside the tile (rows t+1 .. t-3 are all tile rows, no wall event):
// running 32-bit shared addresses, no row-kind branches.  Bit-identical arithmetic to wf_tick.
template <int K>
__device__ __forceinline__ void wf_tick_steady(const int t, WfRegs<K>& R, WfCtx<K>& C, double* __restrict__ sm,
                                               const double* __restrict__ tab)
{
    const WkGeo& g = C.g;
    const int lj = t - g.gys;
    constexpr uint32_t P8 = 8u * WfCtx<K>::P, FS8 = 8u * WfCtx<K>::FS;
    if (C.has_leader && !(t & 1)) {             // (one poll for two ticks: every even tick waits for what the next one needs)
        const int nd = t + 1 + C.dlead < C.TLd + 1 ? t + 1 + C.dlead : C.TLd + 1; wk_wait_prog(C.a_lead, C.need0 + (unsigned)nd);
    }
    if (C.first) wf_wait_xrow<K>(C, lj);
    // ---- loads: own columns of row t, E/W halo and edge u^a of row t-1
    const uint32_t urow = C.sm32 + 8u * (C.st + lj * C.P);          // tile row lj, tile column 0, field 0
    const uint32_t a0 = urow + 8u * (C.c0 - 3), a1 = a0 + FS8, a2 = a1 + FS8;
    double z0[3][K], hz[3][2];
    z0[0][0] = wk_lds<0>(a0); z0[1][0] = wk_lds<0>(a1); z0[2][0] = wk_lds<0>(a2);
    if (K > 1) { z0[0][1] = wk_lds<8>(a0); z0[1][1] = wk_lds<8>(a1); z0[2][1] = wk_lds<8>(a2); }
    if (K > 2) { z0[0][2] = wk_lds<16>(a0); z0[1][2] = wk_lds<16>(a1); z0[2][2] = wk_lds<16>(a2); }
    hz[0][0] = wk_lds<-8>(a0 - P8); hz[1][0] = wk_lds<-8>(a1 - P8); hz[2][0] = wk_lds<-8>(a2 - P8);
    hz[0][1] = wk_lds<8 * K>(a0 - P8); hz[1][1] = wk_lds<8 * K>(a1 - P8); hz[2][1] = wk_lds<8 * K>(a2 - P8);
    const uint32_t ue = urow - P8 + 8u * (g.ex + 3);
    const double eL = wk_lds<0>(ue), eR = wk_lds<8>(ue);
    // ---- stage A on row t-1
    double ha1[K], ua1[K], va1[K];
    {
        const double dtcz1 = tab[t * 8 + WK_T_DTCZ];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double cu = dtcz1 * R.z1[1][i], cv = C.dtcm * R.z1[2][i];
            double xa[3];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double xE = i < K - 1 ? R.z1[f][i + 1 < K ? i + 1 : i] : hz[f][1];
                const double xW = i > 0 ? R.z1[f][i > 0 ? i - 1 : 0] : hz[f][0];
                xa[f] = mm_stageA(R.z1[f][i], xE, xW, z0[f][i], R.z2[f][i], cu, cv, C.kap);
            }
            ha1[i] = xa[0]; ua1[i] = xa[1]; va1[i] = xa[2];
        }
    }
    double uaL1 = wk_up(ua1[K - 1]), uaR1 = wk_dn(ua1[0]);
    uaL1 = C.injL ? eL : uaL1;
    uaR1 = C.injR ? eR : uaR1;
    // ---- h^1 and u^1 on row t-2
    double h12[K], u12[K];
    {
        const double* tb = tab + t * 8 - 8;
        const double dtcz2 = tb[WK_T_DTCZ], gdtcz2 = tb[WK_T_GDTCZ], dtf2 = tb[WK_T_DTF], dtt2 = tb[WK_T_DTT];
        const double rp2 = tb[WK_T_RP], rm2 = tb[WK_T_RM];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double uE = i < K - 1 ? R.ua2[i + 1 < K ? i + 1 : i] : R.uaR2;
            const double uW = i > 0 ? R.ua2[i > 0 ? i - 1 : 0] : R.uaL2;
            h12[i] = mm_h1(R.ha2[i], mm_div(uE, uW, va1[i], R.va3[i], dtcz2, C.dtcm, rp2, rm2));
        }
        const double hL = wk_up(h12[K - 1]), hR = wk_dn(h12[0]);
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double hE = i < K - 1 ? h12[i + 1 < K ? i + 1 : i] : hR;
            const double hW = i > 0 ? h12[i > 0 ? i - 1 : 0] : hL;
            u12[i] = mm_u1(R.ua2[i], R.va2[i], hE, hW, gdtcz2, dtf2, dtt2);
        }
    }
    // ---- v^1 on row t-3 -> row t-3 of Z^{n+1}
    {
        const double dtf3 = tab[t * 8 - 16 + WK_T_DTF], dtt3 = tab[t * 8 - 16 + WK_T_DTT];
        const uint32_t o0 = a0 - 3u * P8, o1 = o0 + FS8, o2 = o1 + FS8;
        double v1[K];
#pragma unroll
        for (int i = 0; i < K; ++i) v1[i] = mm_v1(R.va3[i], R.u13[i], h12[i], R.h14[i], C.gdtcm, dtf3, dtt3);
        if (C.tmask & 1u) { wk_sts<0>(o0, R.h13[0]); wk_sts<0>(o1, R.u13[0]); wk_sts<0>(o2, v1[0]); }
        if (K > 1 && (C.tmask & 2u)) { wk_sts<8>(o0, R.h13[K > 1 ? 1 : 0]); wk_sts<8>(o1, R.u13[K > 1 ? 1 : 0]); wk_sts<8>(o2, v1[K > 1 ? 1 : 0]); }
        if (K > 2 && (C.tmask & 4u)) { wk_sts<16>(o0, R.h13[K > 2 ? 2 : 0]); wk_sts<16>(o1, R.u13[K > 2 ? 2 : 0]); wk_sts<16>(o2, v1[K > 2 ? 2 : 0]); }
        wk_fence_async();
    }
    // ---- E/W ghost cells and edge u^a of row t+1 next to its tile row
    const int l1 = lj + 1, l3 = lj - 3;
    {
        const int slot = (l1 / WK_EWC) & 1, lr = l1 % WK_EWC;
        if (lr == 0) { wk_mbar_wait32(C.b_ew + 8u * slot, (C.par >> (1 + slot)) & 1u); C.par ^= 2u << slot; }
        if (C.lane < 20) {
            const double gv = wk_lds<0>(C.sm32 + 8u * (C.gcp_base + slot * C.gcp_ss + lr * C.gcp_rs));
            wk_sts<0>(urow + P8 + 8u * C.gcp_dst, gv);
        }
    }
    __syncwarp();
    // ---- one lane: progress word, trajectory stores, next E/W chunk
    if (wk_elect()) {
        wk_wait_read<2>();
        wk_publish(C.a_mine, C.gs10 + (unsigned)t + 1u);
        const uint32_t src = urow - 3u * P8;
        double* dst = C.tout + l3 * g.ex;
        wk_s2g32(dst, src, g.ex * 8u); wk_s2g32(dst + g.ncell, src + FS8, g.ex * 8u); wk_s2g32(dst + 2 * g.ncell, src + 2u * FS8, g.ex * 8u);
        wk_commit();
        if ((l1 % WK_EWC) == WK_EWC - 1 && l1 / WK_EWC + 2 < C.nchunk) wf_issue_chunk(C, l1 / WK_EWC + 2);
        if (C.first && lj + WK_XD < g.ey) wf_issue_xrow<K>(C, lj + WK_XD);
    }
    // ---- rotate the row histories
#pragma unroll
    for (int i = 0; i < K; ++i) {
#pragma unroll
        for (int f = 0; f < 3; ++f) { R.z2[f][i] = R.z1[f][i]; R.z1[f][i] = z0[f][i]; }
        R.ha2[i] = ha1[i]; R.ua2[i] = ua1[i]; R.va3[i] = R.va2[i]; R.va2[i] = va1[i];
        R.h14[i] = R.h13[i]; R.h13[i] = h12[i]; R.u13[i] = u12[i];
    }
    R.uaL2 = uaL1; R.uaR2 = uaR1;
}

template <int K>
__global__ void __launch_bounds__(WK_NT, 1) wk_forward(const __grid_constant__ WkArgs A)
{
    extern __shared__ __align__(128) double sm[];
    const int tid = threadIdx.x, lane = tid & 31, w = wk_uni(wk_logical_warp(tid >> 5));
    const WkLayout& Ly = A.Lf;
    const uint32_t sm32 = wk_s32(sm);
    const int IW = Ly.wbase + w * Ly.wsz;
    if (tid == 0) {
        for (int i = 0; i < WK_NW * WK_BAR_PER_WARP; ++i) wk_mbar_init32(sm32 + 8u * i, 1);
        wk_fence_mbar_init();
    }
    if (tid < WK_NW) reinterpret_cast<unsigned*>(sm + WK_PROG)[tid] = 0u;
    for (int q = tid; q < Ly.total - WK_HDR; q += WK_NT) sm[WK_HDR + q] = 0.0;      // no stale NaN patterns
    __syncthreads();                            // the only CTA-wide barrier
    const int lw = (w + WK_NW - 1) % WK_NW;     // the warp that runs the previous step

    WfCtx<K> C;
    C.st = Ly.st;                               // (Ly.P, Ly.FS: compile-time constants of K)
    C.I_SN = IW + Ly.sn; C.I_EW = IW + Ly.ew; C.I_EDS = IW + Ly.eds; C.I_EDE = IW + Ly.ede;
    C.sm32 = sm32; C.a_lead = sm32 + 8u * WK_PROG + 4u * lw; C.a_mine = sm32 + 8u * WK_PROG + 4u * w;
    C.b_sn = sm32 + 8u * (w * WK_BAR_PER_WARP); C.b_ew = C.b_sn + 8u; C.b_x = C.b_sn + 32u;
    C.c0 = 2 + K * lane; C.lane = lane;
    C.kap = A.m.kap; C.dtcm = A.m.dtcm; C.gdtcm = A.m.gdtcm;
    C.A = &A; C.par = 0u;
    constexpr int FS = WfCtx<K>::FS;

    // Every warp walks the same list of (subdomain, step) pairs; global step number gs (1, 2, ...) belongs
    // to warp (gs - 1) % WK_NW, and the step gs - 1 is its leader whatever subdomain it belongs to.
    int nord = -1;                              // ordinal of the current subdomain in this CTA's list
    unsigned gnext = 1u, glast = 0u;            // global numbers: step 0 of the current subdomain, last step of the previous one                        // global number of step 0 of the current subdomain
    int TL = 0, gysL = 0;                       // ticks and south ghost rows of the previous subdomain of this CTA
    for (int k = blockIdx.x; k < A.nsub; k += gridDim.x) {
        if (A.mask && !A.mask[k]) continue;
        ++nord;
        const Sub s = A.subs[k];
        const WkGeo g = wk_geo(s);
        const int T = g.py + 3 - g.gyn;         // the last tile row (padded row py - 1 - gyn) leaves the pipeline three ticks after it enters
        const int n0 = (int)((unsigned)(w + 1) - gnext) & (WK_NW - 1);      // my first step in this subdomain
        if (n0 < g.W) {
            C.g = g; C.T = T;
            // ---------------- per-lane column map of this tile
            C.tmask = 0u;
#pragma unroll
            for (int i = 0; i < K; ++i) if ((C.c0 + i >= 3) && (C.c0 + i < 3 + g.ex)) C.tmask |= 1u << i;
            C.injL = lane == 0; C.injR = (lane == 31) && (C.c0 + K == g.px - 2);
            if (lane < 18) {                    // E/W ghost cell (field lane/6, cell lane%6) of a tile row
                const int f = lane / 6, e = lane % 6;
                C.gcp_base = C.I_EW + f * 6 * WK_EWC + e; C.gcp_ss = 18 * WK_EWC; C.gcp_rs = 6;
                C.gcp_dst = f * FS + (e < 3 ? e - 3 : g.ex + e - 3);
            } else {                            // lanes 18, 19: edge u^a west / east -> the row's two pad cells
                C.gcp_base = C.I_EDE + (lane - 18); C.gcp_ss = 2 * WK_EWC; C.gcp_rs = 2;
                C.gcp_dst = g.ex + 3 + (lane - 18);
            }
            C.nchunk = (g.ey + WK_EWC - 1) / WK_EWC;
            C.xk = A.x + s.coff;
            const double* tab = sm + Ly.tab + (nord % WK_NTAB) * WK_TABSZ(A.maxpy);
        // ---------------- the steps of this warp
        for (int n = n0; n < g.W; n += WK_NW) {
            const unsigned gs = gnext + (unsigned)n;
            C.first = n == 0;
            // the leader: the step before this one, for a first step the last step of the previous subdomain
            const unsigned gl = C.first ? glast : gs - 1u;
            C.gs10 = gs << 10; C.need0 = gl << 10; C.has_leader = gl != 0u;
            C.a_lead = sm32 + 8u * WK_PROG + 4u * ((gl - 1u) & (WK_NW - 1));
            // A first step only OVERWRITES what the previous subdomain left: tile row l is free once that
            // subdomain's last step has stored it and the store has left shared memory (its tick l + gysL + 6).
            C.dlead = C.first ? 7 + WK_XD + gysL - g.gys : 4;
            C.TLd = C.first ? TL : T;
            C.gz = A.ghost + s.goff + (long long)n * 3 * g.nring;
            C.ge = A.gedge + s.eoff + (long long)n * 2 * g.py;
            C.tout = A.traj + s.toff + (long long)(n + 1) * 3 * g.ncell;
            if (wk_elect()) {
                if (g.gys) wf_issue_ns(C, false); else if (g.gyn) wf_issue_ns(C, true);
                wf_issue_chunk(C, 0);
                if (C.nchunk > 1) wf_issue_chunk(C, 1);
            }
            WfRegs<K> R;
#pragma unroll
            for (int i = 0; i < K; ++i) {
#pragma unroll
                for (int f = 0; f < 3; ++f) { R.z1[f][i] = 0.0; R.z2[f][i] = 0.0; }
                R.ha2[i] = R.ua2[i] = R.va2[i] = R.va3[i] = R.h13[i] = R.h14[i] = R.u13[i] = 0.0;
            }
            R.uaL2 = R.uaR2 = 0.0; R.pa = C.I_SN + 1; R.pfs = 0; R.pe = C.I_EDS;

            if (C.first || g.gys == 0) {
                // what tick -1 would do: the control rows that ticks 0 and 1 read, the ghost cells of tile row 0
                if (C.has_leader) { const int nd = C.dlead - 1 < C.TLd + 1 ? C.dlead - 1 : C.TLd + 1; wk_wait_prog(C.a_lead, C.need0 + (unsigned)nd); }
                if (C.first) {
                    wk_copy_tab(sm + Ly.tab + (nord % WK_NTAB) * WK_TABSZ(A.maxpy), A.wtab + (long long)s.b * A.wtab_stride, g.py, lane);
                    wk_fence_async();
                    if (wk_elect())
                        for (int l = 0; l <= WK_XD - 1 - g.gys && l < g.ey; ++l) wf_issue_xrow<K>(C, l);
                }
                if (g.gys == 0) wf_prep_row<K>(C, sm, 0);
                __syncwarp();
            }
            // steady ticks: rows t-3 .. t+1 are tile rows and no wall event falls on the tick
            int ts0 = g.gys + 3; if (ts0 < 4) ts0 = 4;
            const int ts1 = g.gys + g.ey - 1;
#pragma unroll 1
            for (int t = 0; t < C.T;) {
                if (t >= ts0 && t + 1 <= ts1) {
                    wf_tick_steady<K>(t, R, C, sm, tab);
                    t += 1;
                    const int rowb = C.st + (t - 1 - g.gys) * C.P;
                    R.pa = rowb - 3 + C.c0; R.pfs = C.FS; R.pe = rowb + g.ex + 3;
                } else {
                    wf_tick<K>(t, R, C, sm, tab);
                    ++t;
                }
            }
            // step done: all its stores have left shared memory
            if (wk_elect()) { wk_wait_read<0>(); wk_publish(C.a_mine, C.gs10 + (unsigned)C.T + 1u); }
            __syncwarp();
        }
        }
        glast = gnext + (unsigned)g.W - 1u;
        gnext = glast + 1u;
        TL = T; gysL = g.gys;
    }
}
