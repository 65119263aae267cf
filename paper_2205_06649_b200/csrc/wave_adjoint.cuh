// wave_adjoint.cuh -- adjoint sweep of every subdomain (step a4) and the gradient of J_ji at the window
// start, in ONE kernel; see wave_common.cuh for the design and wave_forward.cuh for the tick protocol.
//
// Warp w of the CTA runs adjoint steps m = w, w + WK_NW, ... (m-th step: lambda^n -> lambda^{n-1},
// n = W - m; eq (3)-(4) l.91-98: the window adjoint is the product of the step adjoints in reverse).
// Resident in shared memory, updated IN PLACE row by row: lambda [3][ey][32 K] (zero outside the
// extended tile, so ghost cells are never stored) and u^n [ey][32 K] (the step needs u^1 = u^n of the
// forward step it transposes; the warp of step m leaves u^{n-1}, which it reads anyway, for the
// warp of step m+1).  The linearisation state Z^{n-1} (trajectory store + frozen ghost ring) arrives
// through TMA bulk copies in a per-warp ring of three padded rows.
//
// The step adjoint is the transpose of Phi (model_math.cuh) about Z^{n-1}, evaluated row by row.
// Tick t works on three rows at once (software pipeline inside the warp):
//   row t-1:  stage A recomputed (h^a, u^a, v^a and the differences x_N - x_S); UB, HB, P; and every
//             part of A_h, A_u, A_v that does not need row t:
//               A_u                                   (complete: it only uses row t-1)
//               e   = 1 - dtcz (u^a_E - u^a_W) + dtcm r- v^a_S        (A_h = HB (e - dtcm r+ v^a_N))
//               avp = vb + UB (dtf + dtt u^a) + dtcm r+_{j-1} P_S     (A_v = avp - dtcm r-_{j+1} P_N)
//   row t-2:  A_h, A_v completed with v^a and P of row t-1; L0 in SCATTER form: A(row t-2) adds its
//             centre and east/west parts to row t-2, its southward part to row t-3 (which is then
//             complete and stored) and starts row t-1 with its northward part.  All coefficients of
//             the scatter are local to row t-2 (c_u = dtcz u0, c_v = dtcm v0), so only products
//             cross lanes (shuffles).
// Every row history has depth one or two, so a group of six ticks returns every value to the register it
// started in: the steady loop (rows well inside the tile) is unrolled by six with compile-time slots and
// has no register moves, no row-kind branches and immediate shared-memory offsets.  The remaining
// ticks (ghost rows, pole walls, tails) run the same code with the uniform row-kind tests switched on,
// at slot 0, followed by an explicit rotation.
// Continuous pipeline (wave_common.cuh): the first adjoint step of a subdomain (level W) follows the last
// step of the previous subdomain of this CTA; its input rows lambda^W = 2 mu (Z^W - x_succ) / sigma_b^2 (written
// by ck_cost) and u^W arrive from global memory two ticks ahead, straight into the resident rows.  The last
// step (level 1 -> 0) adds lambda^0 to the control-level part of the gradient that ck_cost left in gx.
// Reflective pole walls (R4): mirrored virtual rows -1 / py as in model_math.cuh; in
// scatter form the part that would leave through the wall comes back into the edge row with the
// sign of the mirrored field.
#pragma once
#include "wave_common.cuh"


template <int K> struct WaState {     // every history has depth one: slot [t & 1] is written at tick t and read at tick t + 1
    double zc[2][3][K];             // [slot][field][column]: Z^{n-1} row t-1 (own columns), kept for one tick as row t-2
    double hz[2][3][2];             // E/W halo of rows t-1, t-2
    double dn[2][3][K];             // x_N - x_S on rows t-1, t-2
    double va[2][K], P[2][K], e[2][K], HB[2][K], Au[2][K], avp[2][K];   // rows t-1, t-2
    double mN[2][3][K];             // northward part of the scatter from row t-2: starts L0 of row t-1
    double La[2][3][K];             // L0 of row t-2 without the southward part of row t-1
};
template <int K> struct WaCtx {
    WkGeo g;
    static constexpr int ZP = WK_AZP(K), FS = WK_AFS(K), maxey = WK_AROWS(K);   // ring row pitch, field stride, zero row
    static constexpr uint32_t SL8 = 24u * ZP, ZP8 = 8u * ZP, FS8 = 8u * FS;      // strides in bytes
    int lam, u1, I_ZR, I_EW, I_EDS, I_EDE, T;
    uint32_t sm32, a_lead, a_mine, b_z, b_ew;
    uint32_t zl, zu, la0;           // per-lane ring / lambda base addresses (shared window)
    unsigned gs10, need0;
    bool has_leader, have_obs, injL, injR, lane0, laneL;    // lane0 / laneL: first lane, lane 31
    bool first, last;               // adjoint step of level W (its input rows arrive from global memory) / of level 1 (its output is the gradient)
    int dlead, TLd;                 // tick t starts when the leader has published min(t + dlead, TLd + 1)
    const double *lw, *uw;          // per lane: lambda^W (ck_cost) and u^W (trajectory store) of own cell 0, tile row 0, field 0
    double* gxl;                    // per lane: gradient cell of own cell 0, tile row 0, field 0
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
    uint32_t dst = C.zu + slot * C.SL8;
    const int lj = r - g.gys;
    const double* src; uint32_t bytes; long long fstride;
    if ((unsigned)lj < (unsigned)g.ey) { src = C.tz + lj * g.ex; bytes = g.ex * 8u; fstride = g.ncell; dst += 32u; }
    else { src = C.gz + (lj < 0 ? r : g.gys + lj - g.ey) * g.px; bytes = g.px * 8u; fstride = g.nring; }
    wk_mbar_expect32(bar, 3u * bytes + (with_edges ? (uint32_t)(g.gys + g.gyn) * 16u : 0u));
    wk_g2s32(dst, src, bytes, bar); wk_g2s32(dst + C.ZP8, src + fstride, bytes, bar); wk_g2s32(dst + 2u * C.ZP8, src + 2 * fstride, bytes, bar);
    if (with_edges && g.gys) wk_g2s32(C.sm32 + 8u * C.I_EDS, C.ge, g.gys * 16u, bar);
    if (with_edges && g.gyn) wk_g2s32(C.sm32 + 8u * (C.I_EDS + 8), C.ge + g.gys * 2, g.gyn * 16u, bar);
}
template <int K>
__device__ __forceinline__ void wa_issue_chunk(const WaCtx<K>& C, int c)
{
    const WkGeo& g = C.g;
    const int r0 = c * WK_EWCA;
    const int rows = g.ey - r0 < WK_EWCA ? g.ey - r0 : WK_EWCA;
    const int slot = c & 1;
    const uint32_t bar = C.b_ew + 8u * slot;
    wk_mbar_expect32(bar, (uint32_t)rows * (3u * 48u + 16u));
    const double* src = C.gz + (g.gys + g.gyn) * g.px + r0 * 6;
    uint32_t dst = C.sm32 + 8u * (C.I_EW + slot * 18 * WK_EWCA);
#pragma unroll 1
    for (int f = 0; f < 3; ++f) { wk_g2s32(dst, src, rows * 48u, bar); dst += 8u * 6 * WK_EWCA; src += g.nring; }
    wk_g2s32(C.sm32 + 8u * (C.I_EDE + slot * 2 * WK_EWCA), C.ge + (g.gys + g.gyn) * 2 + r0 * 2, rows * 16u, bar);
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
        const int cs = (l / WK_EWCA) & 1, lr = l % WK_EWCA;
        if (lr == 0) { wk_mbar_wait32(C.b_ew + 8u * cs, (C.par >> (3 + cs)) & 1u); C.par ^= 8u << cs; }
        if (C.lane < 20) sm[C.I_ZR + slot * 3 * C.ZP + C.gcp_dst] = sm[C.gcp_base + cs * C.gcp_ss + lr * C.gcp_rs];
    }
}

// first adjoint step of a subdomain: tile row l of lambda^W and u^W -> the resident rows (every lane its own
// cells: 8-byte asynchronous copies for tile columns, zeros elsewhere); one cp.async group per call
template <int K>
__device__ __forceinline__ void wa_issue_lamrow(const WaCtx<K>& C, int l)
{
    if ((unsigned)l < (unsigned)C.g.ey) {
        const uint32_t d0 = C.la0 + (uint32_t)l * (8u * 32u * K);
        const double* a = C.lw + l * C.g.ex;
        const double* u = C.uw + l * C.g.ex;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const uint32_t d = d0 + 8u * i;
            if ((C.tmask >> i) & 1u) {
                wk_cpa8(d, a + i); wk_cpa8(d + C.FS8, a + C.g.ncell + i); wk_cpa8(d + 2u * C.FS8, a + 2 * C.g.ncell + i);
                wk_cpa8(d + 3u * C.FS8, u + i);
            } else {
                wk_sts<0>(d, 0.0); wk_sts<0>(d + C.FS8, 0.0); wk_sts<0>(d + 2u * C.FS8, 0.0); wk_sts<0>(d + 3u * C.FS8, 0.0);
            }
        }
    }
    wk_cpa_commit();
}

#define WA_E(arr, i, edge) ((i) < K - 1 ? (arr)[(i) + 1 < K ? (i) + 1 : (i)] : (edge))
#define WA_W(arr, i, edge) ((i) > 0 ? (arr)[(i) > 0 ? (i) - 1 : 0] : (edge))

// One tick.  P2: register slot written by this tick (the other one holds the values of the last tick).
// WALL = false: no pole-wall event falls on this tick (every tick of a tile without walls; on such
// ticks whatever is computed on rows outside the padded tile is finite and multiplies lambda = 0).
template <int K, int P2, bool WALL>
__device__ __forceinline__ void wa_tick(const int t, WaState<K>& S, WaCtx<K>& C, double* __restrict__ sm,
                                        const double* __restrict__ tab)
{
    constexpr int pn = P2, po = 1 - P2;
    constexpr uint32_t PL8 = 8u * 32u * K;          // lambda row pitch in bytes
    const WkGeo& g = C.g;
    const int lj = t - g.gys;
    const bool tile = (unsigned)lj < (unsigned)g.ey;
    const bool tile1 = (unsigned)(lj - 1) < (unsigned)g.ey;
    double zN[3][K];                                // row t (re-read as row t-1 by the next tick: the ring still holds it)
    double (&zC)[3][K] = S.zc[pn];
    double (&zS)[3][K] = S.zc[po];
    // ---- (0) the leader has finished row t of lambda^n and u^n; H^T R^-1 (25b) forcing on that row.  First in the tick:
    // the read-modify-write of the forcing and the first step's row copies complete behind stages (1) and (2a), which
    // work on the warp's private ring (4.43 -> 4.33 ms against the poll after stage (2a); one poll per pair of ticks: 4.29 ms)
    if (C.has_leader && (WALL || P2 == 0)) {        // (a pair of ticks: one poll, for what the second tick needs)
        const int nd = t + 1 + C.dlead < C.TLd + 1 ? t + 1 + C.dlead : C.TLd + 1;
        wk_wait_prog(C.a_lead, C.need0 + (unsigned)nd);
    }
    if (C.first) {                                  // row t of lambda^W / u^W has landed; fetch row t + 2
        wk_cpa_wait<1>();
        wa_issue_lamrow<K>(C, lj + 2);
        __syncwarp();
    }
    if (tile && C.have_obs) {
        const WkArgs& A = *C.A;
        for (;;) {
            const unsigned mm = __ballot_sync(0xffffffffu, (C.p_pk >> 12) == lj);
            const int cnt = __popc(mm);
            if (cnt == 0) break;
            if (C.lane < cnt) sm[C.lam + ((C.p_pk >> 8) & 3) * C.FS + lj * (32 * K) + 1 + (C.p_pk & 255)] += C.p_r;
            C.qcur += cnt;
            C.p_pk = 0x7fffffff;
            if (C.qcur + C.lane < C.qend) { C.p_pk = A.obs_lj[C.qcur + C.lane]; C.p_r = A.obs_r[C.qcur + C.lane]; }
            if (cnt < 32) break;
        }
        __syncwarp();
    }
    // ---- (1) Z^{n-1}: own columns of row t, E/W halo and edge u^a of row t-1
    double eL, eR;
    {
        const int s0 = t % 3, s1 = s0 == 0 ? 2 : s0 - 1;             // ring slots of rows t, t-1
        const uint32_t h0 = C.zl + s1 * C.SL8 + (tile1 ? 8u : 0u), h1 = h0 + C.ZP8, h2 = h1 + C.ZP8;
        if (!WALL || t <= g.py) {                   // row t-1 is a padded row (at t = 0: stale but finite data)
            zC[0][0] = wk_lds<0>(h0); zC[1][0] = wk_lds<0>(h1); zC[2][0] = wk_lds<0>(h2);
            if (K > 1) { zC[0][K > 1 ? 1 : 0] = wk_lds<8>(h0); zC[1][K > 1 ? 1 : 0] = wk_lds<8>(h1); zC[2][K > 1 ? 1 : 0] = wk_lds<8>(h2); }
            if (K > 2) { zC[0][K > 2 ? 2 : 0] = wk_lds<16>(h0); zC[1][K > 2 ? 2 : 0] = wk_lds<16>(h1); zC[2][K > 2 ? 2 : 0] = wk_lds<16>(h2); }
        } else {
#pragma unroll
            for (int i = 0; i < K; ++i) { zC[0][i] = zS[0][i]; zC[1][i] = zS[1][i]; zC[2][i] = zS[2][i]; }
        }
        if (!WALL || t < g.py) {
            const uint32_t a0 = C.zl + s0 * C.SL8 + (tile ? 8u : 0u), a1 = a0 + C.ZP8, a2 = a1 + C.ZP8;
            zN[0][0] = wk_lds<0>(a0); zN[1][0] = wk_lds<0>(a1); zN[2][0] = wk_lds<0>(a2);
            if (K > 1) { zN[0][K > 1 ? 1 : 0] = wk_lds<8>(a0); zN[1][K > 1 ? 1 : 0] = wk_lds<8>(a1); zN[2][K > 1 ? 1 : 0] = wk_lds<8>(a2); }
            if (K > 2) { zN[0][K > 2 ? 2 : 0] = wk_lds<16>(a0); zN[1][K > 2 ? 2 : 0] = wk_lds<16>(a1); zN[2][K > 2 ? 2 : 0] = wk_lds<16>(a2); }
        } else {
            const double sg = (t == g.py && g.wn) ? -1.0 : 1.0;     // virtual mirrored row py
#pragma unroll
            for (int i = 0; i < K; ++i) { zN[0][i] = zC[0][i]; zN[1][i] = zC[1][i]; zN[2][i] = sg * zC[2][i]; }
        }
        S.hz[pn][0][0] = wk_lds<-8>(h0); S.hz[pn][1][0] = wk_lds<-8>(h1); S.hz[pn][2][0] = wk_lds<-8>(h2);
        S.hz[pn][0][1] = wk_lds<8 * K>(h0); S.hz[pn][1][1] = wk_lds<8 * K>(h1); S.hz[pn][2][1] = wk_lds<8 * K>(h2);
        uint32_t ea, eb;
        if (tile1) { ea = C.zu + s1 * C.SL8; eb = ea + C.ZP8; }
        else {
            const int l1 = lj - 1;
            ea = C.sm32 + 8u * (uint32_t)(C.I_EDS + (l1 >= g.ey ? 8 + (l1 - g.ey) * 2 : (t > 0 ? (t - 1) * 2 : 0)));
            eb = ea + 8u;
        }
        eL = wk_lds<0>(ea); eR = wk_lds<0>(eb);
    }
    if (WALL && g.ws && t == 1) {                   // virtual row -1 (R4)
#pragma unroll
        for (int i = 0; i < K; ++i) { zS[0][i] = zC[0][i]; zS[1][i] = zC[1][i]; zS[2][i] = -zC[2][i]; }
    }
    const bool stage2 = WALL ? t <= g.py : true;    // row t-1 is a padded row
    const bool vrN = WALL ? (g.wn && t == g.py + 1) : false;     // row t-1 is the virtual row py
    const double* t1 = tab + t * 8;                 // table entry of row t-1
    const double* t2 = tab + (t > 0 ? t - 1 : 0) * 8;      // row t-2

    // ---- (2a) row t-1: stage A recomputed
    double ha1[K], ua1[K], uaW, uaE;
    if (stage2) {
        const double dtcz1 = t1[WK_T_DTCZ];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double cu = dtcz1 * zC[1][i], cv = C.dtcm * zC[2][i];
            double xa[3];
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                const double xE = WA_E(zC[f], i, S.hz[pn][f][1]);
                const double xW = WA_W(zC[f], i, S.hz[pn][f][0]);
                const double dnf = zN[f][i] - zS[f][i];
                S.dn[pn][f][i] = dnf;
                xa[f] = zC[f][i] - (cu * (xE - xW) + cv * dnf) + C.kap * (xE + xW + zN[f][i] + zS[f][i] - 4.0 * zC[f][i]);
            }
            ha1[i] = xa[0]; ua1[i] = xa[1]; S.va[pn][i] = xa[2];
        }
        uaW = wk_up(ua1[K - 1]); uaE = wk_dn(ua1[0]);
        uaW = C.injL ? eL : uaW; uaE = C.injR ? eR : uaE;     // frozen u^a of the ghost columns 1 and px-2 (xk_edge_ua)
    } else {
#pragma unroll
        for (int i = 0; i < K; ++i) {
            ha1[i] = 0.0; ua1[i] = 0.0; S.va[pn][i] = vrN ? -S.va[po][i] : 0.0;     // virtual row py: v^a mirrored
#pragma unroll
            for (int f = 0; f < 3; ++f) S.dn[pn][f][i] = 0.0;
        }
        uaW = 0.0; uaE = 0.0;
    }
    // ---- (2b) lambda^n: v rows t, t-1, t-2; h, u and u^n row t-1.  UB, HB, P and the row-local parts of A on row t-1
    const uint32_t lrow = C.la0 + (uint32_t)lj * PL8;      // own cell 0 of lambda_h, tile row lj (may lie outside the tile)
    double P1[K];
    if (stage2) {
        const uint32_t zrow = C.la0 + (uint32_t)C.maxey * PL8;          // the all-zero row
        const uint32_t ah = tile1 ? lrow - PL8 : zrow, au = ah + C.FS8, a1 = ah + 3u * C.FS8, ac = ah + 2u * C.FS8;
        const double dtcz1 = t1[WK_T_DTCZ], gdtcz1 = t1[WK_T_GDTCZ], dtf1 = t1[WK_T_DTF], dtt1 = t1[WK_T_DTT];
        const double cmrm1 = t1[WK_T_CMRM], cmrp2 = t2[WK_T_CMRP];
        double hb1[K], ub1[K], u1r[K], vbN[K], vbC[K], vbS[K];
        {
            // (rows t-1 and t-2 of lambda_v are still in place: row r is overwritten at tick r + 3)
            const bool tile2 = (unsigned)(lj - 2) < (unsigned)g.ey;
            const uint32_t av = (tile ? lrow : zrow) + 2u * C.FS8, as = (tile2 ? lrow - 2u * PL8 : zrow) + 2u * C.FS8;
            vbN[0] = wk_lds<0>(av); hb1[0] = wk_lds<0>(ah); ub1[0] = wk_lds<0>(au); u1r[0] = wk_lds<0>(a1);
            vbC[0] = wk_lds<0>(ac); vbS[0] = wk_lds<0>(as);
            if (K > 1) { vbN[K > 1 ? 1 : 0] = wk_lds<8>(av); hb1[K > 1 ? 1 : 0] = wk_lds<8>(ah); ub1[K > 1 ? 1 : 0] = wk_lds<8>(au); u1r[K > 1 ? 1 : 0] = wk_lds<8>(a1);
                         vbC[K > 1 ? 1 : 0] = wk_lds<8>(ac); vbS[K > 1 ? 1 : 0] = wk_lds<8>(as); }
            if (K > 2) { vbN[K > 2 ? 2 : 0] = wk_lds<16>(av); hb1[K > 2 ? 2 : 0] = wk_lds<16>(ah); ub1[K > 2 ? 2 : 0] = wk_lds<16>(au); u1r[K > 2 ? 2 : 0] = wk_lds<16>(a1);
                         vbC[K > 2 ? 2 : 0] = wk_lds<16>(ac); vbS[K > 2 ? 2 : 0] = wk_lds<16>(as); }
        }
        if (WALL && g.ws && t == 1) {               // virtual row -1: lambda_v mirrored
#pragma unroll
            for (int i = 0; i < K; ++i) vbS[i] = -vbC[i];
        }
        if (WALL && g.wn && t == g.py) {            // virtual row py: lambda_v mirrored
#pragma unroll
            for (int i = 0; i < K; ++i) vbN[i] = -vbC[i];
        }
        double UB1[K];
#pragma unroll
        for (int i = 0; i < K; ++i) UB1[i] = mm_UB(ub1[i], vbC[i], u1r[i], dtf1, dtt1);
        double UBW = wk_up(UB1[K - 1]), UBE = wk_dn(UB1[0]);
        UBW = C.lane0 ? 0.0 : UBW; UBE = C.laneL ? 0.0 : UBE;          // ghost columns: lambda = 0
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double hb = mm_HB(hb1[i], vbN[i], vbS[i], WA_E(UB1, i, UBE), WA_W(UB1, i, UBW), C.gdtcm, gdtcz1);
            P1[i] = -ha1[i] * hb;
            S.HB[pn][i] = hb;                       // (HB of row t-2 sits in the other slot until (3) has read it)
        }
        double PW = wk_up(P1[K - 1]), PE = wk_dn(P1[0]);
        PW = C.lane0 ? 0.0 : PW; PE = C.laneL ? 0.0 : PE;
        const bool wS1 = WALL ? (g.ws && t == 1) : false;          // row t-2 is the virtual row -1
        const double rm0 = WALL ? tab[8 + WK_T_RM] : 0.0;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const double vaS = wS1 ? -S.va[pn][i] : S.va[po][i];
            const double PS = wS1 ? rm0 * P1[i] : S.P[po][i];
            S.Au[pn][i] = mm_Au(UB1[i], S.va[pn][i], WA_W(P1, i, PW), WA_E(P1, i, PE), dtt1, dtcz1);
            S.e[pn][i] = 1.0 - dtcz1 * (WA_E(ua1, i, uaE) - WA_W(ua1, i, uaW)) + cmrm1 * vaS;
            S.avp[pn][i] = vbC[i] + UB1[i] * (dtf1 + dtt1 * ua1[i]) + cmrp2 * PS;
        }
    } else {
        const double rpn = tab[g.py * 8 + WK_T_RP];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            P1[i] = vrN ? rpn * S.P[po][i] : 0.0;   // virtual row py: P carries the metric ratio
            S.HB[pn][i] = 0.0; S.Au[pn][i] = 0.0; S.e[pn][i] = 0.0; S.avp[pn][i] = 0.0;
        }
    }
    // ---- (3) row t-2: A_h, A_u, A_v completed; (4) scatter into L0 of rows t-1, t-2, t-3
    double (&Ln)[3][K] = S.mN[pn];                  // L0 of row t-1: northward part of the scatter from row t-2
    double (&La)[3][K] = S.La[pn];                  // L0 of row t-2 (its southward part arrives at the next tick)
    double Lb[3][K];                                // L0 of row t-3: complete
    if (!WALL || (t >= 2 && t <= g.py + 1)) {       // (rows -1 and py are virtual: nothing is scattered from them)
        const double dtcz2 = t2[WK_T_DTCZ], cmrp2 = t2[WK_T_CMRP], cmrm1 = t1[WK_T_CMRM];
        const bool wallS = WALL ? (g.ws && t == 2) : false, wallN = WALL ? (g.wn && t == g.py + 1) : false;
        double Aa[3][K], cu[K], cv[K], su[K], sv[K];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            Aa[0][i] = S.HB[po][i] * (S.e[po][i] - cmrp2 * S.va[pn][i]);
            Aa[1][i] = S.Au[po][i];
            Aa[2][i] = S.avp[po][i] - cmrm1 * P1[i];
            cu[i] = dtcz2 * zS[1][i]; cv[i] = C.dtcm * zS[2][i];
            su[i] = 0.0; sv[i] = 0.0;
        }
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            double mE[K], mW[K];
            const double sgn = f == 2 ? -1.0 : 1.0;
#pragma unroll
            for (int i = 0; i < K; ++i) {
                const double a = Aa[f][i];
                const double xE = WA_E(zS[f], i, S.hz[po][f][1]);
                const double xW = WA_W(zS[f], i, S.hz[po][f][0]);
                mE[i] = a * (C.kap - cu[i]); mW[i] = a * (C.kap + cu[i]);
                su[i] += (xE - xW) * a; sv[i] += S.dn[po][f][i] * a;
                const double mS = a * (C.kap + cv[i]), mN = a * (C.kap - cv[i]);
                double la = S.mN[po][f][i] + a * C.c0k;
                if (wallS) { la += sgn * mS; Lb[f][i] = S.La[po][f][i]; } else Lb[f][i] = S.La[po][f][i] + mS;
                if (wallN) { la += sgn * mN; Ln[f][i] = 0.0; } else Ln[f][i] = mN;
                La[f][i] = la;
            }
            const double fW = wk_up(mE[K - 1]), fE = wk_dn(mW[0]);
#pragma unroll
            for (int i = 0; i < K; ++i) La[f][i] += WA_W(mE, i, fW) + WA_E(mW, i, fE);
        }
#pragma unroll
        for (int i = 0; i < K; ++i) { La[1][i] -= dtcz2 * su[i]; La[2][i] -= C.dtcm * sv[i]; }
    } else {
#pragma unroll
        for (int f = 0; f < 3; ++f)
#pragma unroll
            for (int i = 0; i < K; ++i) { Ln[f][i] = 0.0; La[f][i] = S.mN[po][f][i]; Lb[f][i] = S.La[po][f][i]; }
    }
#pragma unroll
    for (int i = 0; i < K; ++i) S.P[pn][i] = P1[i];
    // ---- (5) row t-3 of lambda^{n-1} is complete; u^{n-1} of row t-2 replaces u^n
    {
        const bool st3 = (unsigned)(lj - 3) < (unsigned)g.ey;
        const bool st2 = (unsigned)(lj - 2) < (unsigned)g.ey;
        const uint32_t o0 = lrow - 3u * PL8, o1 = o0 + C.FS8, o2 = o1 + C.FS8, o3 = lrow - 2u * PL8 + 3u * C.FS8;
        if (st3 && C.last) {
            // lambda^0 of row t-3: added to the control-level part of the gradient ck_cost left in gx
            // (one reduction per cell, no return value: the sum does not depend on timing)
            double* gp = C.gxl + (lj - 3) * g.ex;
#pragma unroll
            for (int i = 0; i < K; ++i)
                if ((C.tmask >> i) & 1u) {
#pragma unroll
                    for (int f = 0; f < 3; ++f) atomicAdd(gp + (long long)f * g.ncell + i, Lb[f][i]);
                }
        } else if (st3) {
            if (C.tmask & 1u) { wk_sts<0>(o0, Lb[0][0]); wk_sts<0>(o1, Lb[1][0]); wk_sts<0>(o2, Lb[2][0]); }
            if (K > 1 && (C.tmask & 2u)) { wk_sts<8>(o0, Lb[0][K > 1 ? 1 : 0]); wk_sts<8>(o1, Lb[1][K > 1 ? 1 : 0]); wk_sts<8>(o2, Lb[2][K > 1 ? 1 : 0]); }
            if (K > 2 && (C.tmask & 4u)) { wk_sts<16>(o0, Lb[0][K > 2 ? 2 : 0]); wk_sts<16>(o1, Lb[1][K > 2 ? 2 : 0]); wk_sts<16>(o2, Lb[2][K > 2 ? 2 : 0]); }
        }
        if (st2 && !C.last) {
            if (C.tmask & 1u) wk_sts<0>(o3, zS[1][0]);
            if (K > 1 && (C.tmask & 2u)) wk_sts<8>(o3, zS[1][K > 1 ? 1 : 0]);
            if (K > 2 && (C.tmask & 4u)) wk_sts<16>(o3, zS[1][K > 2 ? 2 : 0]);
        }
    }
    // the next row of Z^{n-1} must have landed; its ghost cells go in place
    if (t + 1 < g.py) wa_prep_row<K>(C, sm, t + 1);
    __syncwarp();
    // ---- (6) one lane: progress word, the row after next, next E/W chunk
    if (wk_elect()) {
        wk_publish(C.a_mine, C.gs10 + (unsigned)t + 1u);
        if (t + 2 < g.py) wa_issue_row<K>(C, t + 2, false);
        const int l1 = lj + 1;
        if ((unsigned)l1 < (unsigned)g.ey && (l1 % WK_EWCA) == WK_EWCA - 1 && l1 / WK_EWCA + 2 < C.nchunk)
            wa_issue_chunk<K>(C, l1 / WK_EWCA + 2);
    }
}

// after a single tick run at slot 0: move every history to slot 1, where the next tick at slot 0 reads it
template <int K>
__device__ __forceinline__ void wa_rotate(WaState<K>& S)
{
#pragma unroll
    for (int i = 0; i < K; ++i) {
#pragma unroll
        for (int f = 0; f < 3; ++f) {
            S.zc[1][f][i] = S.zc[0][f][i]; S.dn[1][f][i] = S.dn[0][f][i];
            S.mN[1][f][i] = S.mN[0][f][i]; S.La[1][f][i] = S.La[0][f][i];
        }
        S.va[1][i] = S.va[0][i]; S.P[1][i] = S.P[0][i]; S.e[1][i] = S.e[0][i];
        S.HB[1][i] = S.HB[0][i]; S.Au[1][i] = S.Au[0][i]; S.avp[1][i] = S.avp[0][i];
    }
#pragma unroll
    for (int f = 0; f < 3; ++f) { S.hz[1][f][0] = S.hz[0][f][0]; S.hz[1][f][1] = S.hz[0][f][1]; }
}

template <int K>
__global__ void __launch_bounds__(WK_NT, 1) wk_adjoint(const __grid_constant__ WkArgs A)
{
    extern __shared__ __align__(128) double sm[];
    const int tid = threadIdx.x, lane = tid & 31, w = wk_uni(wk_logical_warp(tid >> 5));
    const WkLayout& Ly = A.La;
    const uint32_t sm32 = wk_s32(sm);
    const int IW = Ly.wbase + w * Ly.wsz;
    if (tid == 0) {
        for (int i = 0; i < WK_NW * WK_BAR_PER_WARP; ++i) wk_mbar_init32(sm32 + 8u * i, 1);
        wk_fence_mbar_init();
    }
    if (tid < WK_NW) reinterpret_cast<unsigned*>(sm + WK_PROG)[tid] = 0u;
    for (int q = tid; q < Ly.total - WK_HDR; q += WK_NT) sm[WK_HDR + q] = 0.0;     // (the zero row and the pad cells stay zero)
    __syncthreads();                            // the only CTA-wide barrier
    const int lw = (w + WK_NW - 1) % WK_NW;

    WaCtx<K> C;
    C.lam = Ly.st; C.u1 = Ly.u1;                // (Ly.ZP, Ly.FS: compile-time constants of K, wave_common.cuh)
    C.I_ZR = IW + Ly.zr; C.I_EW = IW + Ly.ew; C.I_EDS = IW + Ly.eds; C.I_EDE = IW + Ly.ede;
    C.sm32 = sm32; C.a_lead = sm32 + 8u * WK_PROG + 4u * lw; C.a_mine = sm32 + 8u * WK_PROG + 4u * w;
    C.b_z = sm32 + 8u * (w * WK_BAR_PER_WARP); C.b_ew = C.b_z + 24u;
    C.c0 = 2 + K * lane; C.lane = lane; C.lane0 = lane == 0; C.laneL = lane == 31;
    C.zu = sm32 + 8u * C.I_ZR; C.zl = C.zu + 8u * C.c0;
    C.la0 = sm32 + 8u * (Ly.st + K * lane);
    C.kap = A.m.kap; C.dtcm = A.m.dtcm; C.gdtcm = A.m.gdtcm; C.c0k = 1.0 - 4.0 * A.m.kap; C.mu2 = 2.0 * A.cp.mu;
    C.A = &A; C.par = 0u;

    // Every warp walks the same list of (subdomain, adjoint step) pairs (see wk_forward).
    int nord = -1;                              // ordinal of the current subdomain in this CTA's list
    unsigned gnext = 1u, glast = 0u;            // global numbers: step 0 of the current subdomain, last step of the previous one
    int TL = 0, gysL = 0;
    for (int k = blockIdx.x; k < A.nsub; k += gridDim.x) {
        if (A.mask && !A.mask[k]) continue;
        ++nord;
        const Sub s = A.subs[k];
        const WkGeo g = wk_geo(s);
        // (tiles without pole walls: an even number of ticks, so that all of them run in pairs and the single-tick body
        //  stays out of the hot loop; the extra tick works on rows beyond the tile, whose lambda is zero, and stores nothing)
        const int T = g.py + 3 - g.gyn + ((!g.ws && !g.wn) ? ((g.py + 3 - g.gyn) & 1) : 0);
        const int m0 = (int)((unsigned)(w + 1) - gnext) & (WK_NW - 1);
        if (m0 < g.W) {
            C.g = g; C.T = T;
            const long long n3 = 3LL * g.ncell;
            // ---------------- per-lane column map of this tile
            C.tmask = 0u;
#pragma unroll
            for (int i = 0; i < K; ++i) if ((C.c0 + i >= 3) && (C.c0 + i < 3 + g.ex)) C.tmask |= 1u << i;
            C.injL = lane == 0; C.injR = (lane == 31) && (C.c0 + K == g.px - 2);
            if (lane < 18) {                    // E/W ghost cell (field lane/6, cell lane%6) -> padded columns 0..2, px-3..px-1
                const int f = lane / 6, e = lane % 6;
                C.gcp_base = C.I_EW + f * 6 * WK_EWCA + e; C.gcp_ss = 18 * WK_EWCA; C.gcp_rs = 6;
                C.gcp_dst = f * C.ZP + 1 + (e < 3 ? e : g.ex + e);
            } else {                            // lanes 18, 19: edge u^a west / east -> the free cell 0 of fields 0 / 1
                C.gcp_base = C.I_EDE + (lane - 18); C.gcp_ss = 2 * WK_EWCA; C.gcp_rs = 2;
                C.gcp_dst = (lane - 18) * C.ZP;
            }
            C.nchunk = (g.ey + WK_EWCA - 1) / WK_EWCA;
            // own cell 0 <-> padded column 2 + K lane <-> tile column K lane - 1
            C.lw = A.lamW + s.coff + (K * lane - 1);
            C.uw = A.traj + s.toff + (long long)g.W * n3 + g.ncell + (K * lane - 1);
            C.gxl = A.gx + s.coff + (K * lane - 1);
            const double* tab = sm + Ly.tab + (nord % WK_NTAB) * WK_TABSZ(A.maxpy);

        // ---------------- the steps of this warp
        for (int m = m0; m < g.W; m += WK_NW) {
            const int n = g.W - m;
            const unsigned gs = gnext + (unsigned)m;
            C.first = m == 0;
            // the leader: the step before this one, for a first step the last step of the previous subdomain
            const unsigned gl = C.first ? glast : gs - 1u;
            C.gs10 = gs << 10; C.need0 = gl << 10; C.has_leader = gl != 0u;
            C.a_lead = sm32 + 8u * WK_PROG + 4u * ((gl - 1u) & (WK_NW - 1)); C.last = n == 1;
            // A first step only OVERWRITES what the previous subdomain left: its last step (which stores nothing in
            // shared memory) has finished with tile row l after its tick l + gysL + 2.
            C.dlead = C.first ? 5 + gysL - g.gys : 4;
            C.TLd = C.first ? TL : T;
            C.gz = A.ghost + s.goff + (long long)(n - 1) * 3 * g.nring;
            C.ge = A.gedge + s.eoff + (long long)(n - 1) * 2 * g.py;
            C.tz = A.traj + s.toff + (long long)(n - 1) * n3;
            C.qcur = 0; C.qend = 0;
            if (A.obs_start && m > 0) { C.qcur = A.obs_start[s.ooff + n]; C.qend = A.obs_start[s.ooff + n + 1]; }   // (level W: its forcing is part of lambda^W, ck_cost / ck_gn)
            C.have_obs = C.qend > C.qcur;
            C.p_pk = 0x7fffffff; C.p_r = 0.0;
            if (C.have_obs && C.qcur + lane < C.qend) { C.p_pk = A.obs_lj[C.qcur + lane]; C.p_r = A.obs_r[C.qcur + lane]; }
            if (wk_elect()) {
                wa_issue_row<K>(C, 0, true);
                if (g.py > 1) wa_issue_row<K>(C, 1, false);
                wa_issue_chunk<K>(C, 0);
                if (C.nchunk > 1) wa_issue_chunk<K>(C, 1);
            }
            WaState<K> S;
#pragma unroll
            for (int sl = 0; sl < 2; ++sl) {
#pragma unroll
                for (int i = 0; i < K; ++i) {
#pragma unroll
                    for (int f = 0; f < 3; ++f) { S.zc[sl][f][i] = 0.0; S.dn[sl][f][i] = 0.0; S.mN[sl][f][i] = 0.0; S.La[sl][f][i] = 0.0; }
                    S.va[sl][i] = S.P[sl][i] = S.e[sl][i] = S.HB[sl][i] = S.Au[sl][i] = S.avp[sl][i] = 0.0;
                }
#pragma unroll
                for (int f = 0; f < 3; ++f) { S.hz[sl][f][0] = 0.0; S.hz[sl][f][1] = 0.0; }
            }
            if (C.first) {
                // what ticks -2 and -1 would do: the rows of lambda^W / u^W that ticks 0 and 1 read
                if (C.has_leader) { const int nd = C.dlead < C.TLd + 1 ? C.dlead : C.TLd + 1; wk_wait_prog(C.a_lead, C.need0 + (unsigned)nd); }
                wk_copy_tab(sm + Ly.tab + (nord % WK_NTAB) * WK_TABSZ(A.maxpy), A.wtab + (long long)s.b * A.wtab_stride, g.py, lane);
                wa_issue_lamrow<K>(C, -g.gys);
                wa_issue_lamrow<K>(C, 1 - g.gys);
            }
            wa_prep_row<K>(C, sm, 0);           // (the ring is private to this warp: no leader involved)
            __syncwarp();
            // ticks [0, tp0) and [tp1, T): one at a time (pole-wall events, odd remainder); ticks [tp0, tp1): in
            // pairs (a pair returns every history to the register slot it started in: no register moves)
            const int tp0 = g.ws ? 3 : 0;
            int tp1 = g.wn ? g.py : C.T;
            tp1 -= (tp1 - tp0) & 1;
            int t = 0;
#pragma unroll 1
            for (int ph = 0; ph < 2; ++ph) {
                const int tend = ph == 0 ? tp0 : C.T;
#pragma unroll 1
                for (; t < tend; ++t) {
                    if ((g.ws && t <= 2) || (g.wn && t >= g.py)) wa_tick<K, 0, true>(t, S, C, sm, tab);
                    else wa_tick<K, 0, false>(t, S, C, sm, tab);
                    wa_rotate<K>(S);
                }
                if (ph == 0) {
#pragma unroll 1
                    for (; t < tp1; t += 2) {
                        wa_tick<K, 0, false>(t, S, C, sm, tab);
                        wa_tick<K, 1, false>(t + 1, S, C, sm, tab);
                    }
                }
            }
            if (C.first) wk_cpa_wait<0>();
            if (wk_elect()) wk_publish(C.a_mine, C.gs10 + (unsigned)C.T + 1u);
            __syncwarp();
        }
        }
        glast = gnext + (unsigned)g.W - 1u;
        gnext = glast + 1u;
        TL = T; gysL = g.gys;
    }
}
