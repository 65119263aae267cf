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
#pragma once
#include "wave_common.cuh"

template <int K>
__global__ void __launch_bounds__(WK_NT, 1) wk_forward(const __grid_constant__ WkArgs A)
{
    extern __shared__ __align__(128) double sm[];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const WkLayout Ly = wk_layout(false, A.maxex, A.maxey, A.maxpx, A.maxpy);
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm);
    uint64_t* bar_sn = bars + w * 5;
    uint64_t* bar_ew = bars + w * 5 + 1;       // [2]
    uint64_t* bar_init = bars + 40;
    const uint32_t a_prog = wk_s32(sm + 48);   // WK_NW progress words (u32)
    int* s_next = reinterpret_cast<int*>(sm + 52);
    double* red = sm + 64;                      // [32] block reduction scratch
    double* wpart = sm + 96;                    // [WK_NW] observation cost of each warp's steps
    double* tab = sm + Ly.tab;
    const int IW = Ly.wbase + w * Ly.wsz;
    const int I_SN = IW + Ly.sn, I_EW = IW + Ly.ew, I_EDS = IW + Ly.eds, I_EDE = IW + Ly.ede;
    if (tid == 0) {
        for (int i = 0; i < 41; ++i) wk_mbar_init(bars + i, 1);
        wk_fence_mbar_init();
    }
    if (tid < WK_NW) reinterpret_cast<unsigned*>(sm + 48)[tid] = 0u;
    __syncthreads();
    unsigned par = 0u, par_init = 0u;           // phase parities: bit 0 sn, bits 1,2 ew slots
    unsigned gbase = 1u;                        // CTA-wide step counter (progress words only grow)
    const int lw = (w + WK_NW - 1) % WK_NW;     // the warp that runs the previous step
    const int c0 = 2 + K * lane;                // first padded column this lane owns
    const double kap = A.m.kap, dtcm = A.m.dtcm, gdtcm = A.m.gdtcm;

    for (;;) {
        if (tid == 0) *s_next = atomicAdd(A.counter, 1);
        __syncthreads();
        const int k = *s_next;
        __syncthreads();
        if (k >= A.nsub) break;
        if (A.mask && !A.mask[k]) continue;
        const Sub s = A.subs[k];
        const WkGeo g = wk_geo(s);
        const int st = Ly.st, P = Ly.P, FS = Ly.FS;

        // ---------------- init: control -> resident state (TMA), row tables, level 0 of the store
        if (tid == 0) wk_mbar_expect(bar_init, 3u * g.ncell * 8u);
        wk_load_tab(tab, A.m, g);
        __syncthreads();
        for (int q = tid; q < 3 * g.ey; q += WK_NT) {
            const int f = q / g.ey, lj = q - f * g.ey;
            wk_g2s(sm + st + f * FS + lj * P, A.x + s.coff + (long long)f * g.ncell + lj * g.ex, g.ex * 8u, bar_init);
        }
        wk_mbar_wait(bar_init, par_init); par_init ^= 1u;
        __syncthreads();
        for (int q = tid; q < 3 * g.ey; q += WK_NT) {
            const int f = q / g.ey, lj = q - f * g.ey;
            wk_s2g(A.traj + s.toff + (long long)f * g.ncell + lj * g.ex, sm + st + f * FS + lj * P, g.ex * 8u);
        }
        wk_commit();

        // ---------------- control-level cost terms: (25a) background, (25c) spatial overlap and
        // predecessor window, and H (25b) at level 0; the successor term follows the sweep
        double bg = 0.0, sp = 0.0, pr = 0.0, ob = 0.0;
        {
            const bool pred = s.jw > 0;
            for (int c = tid; c < g.ncell; c += WK_NT) {
                const int lj = c / g.ex, li = c - lj * g.ex;
                const int gi = imodd(s.ei0 + li, A.geo.nlon), gj = s.ej0 + lj;
                const int nc = A.geo.ncolcov[gi], nr = A.geo.nrowcov[gj];
                const double wsp = 1.0 / (double)(nc * nr);
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    const double xv = sm[st + f * FS + lj * P + li];
                    const double db = xv - A.xbs[s.coff + (long long)f * g.ncell + c];
                    bg += wsp * db * db * A.cp.ib[f];
                    if (nc * nr > 1)
                        for (int cb = 0; cb < nr; ++cb)
                            for (int ca = 0; ca < nc; ++ca) {
                                const int a2 = A.geo.colcov[4 * gi + ca], b2 = A.geo.rowcov[4 * gj + cb];
                                if (a2 == s.a && b2 == s.b) continue;
                                const Sub& s2 = A.subs[(s.jw * A.geo.p2 + b2) * A.geo.p1 + a2];
                                const int li2 = imodd(gi - s2.ei0, A.geo.nlon), lj2 = gj - s2.ej0;
                                const double dv = xv - A.xfrozen[s2.coff + (long long)f * s2.ncell + lj2 * s2.ex + li2];
                                sp += dv * dv * A.cp.ib[f];
                            }
                    if (pred) {
                        const double dv = xv - A.pred_end[s.coff + (long long)f * g.ncell + c];
                        pr += dv * dv * A.cp.ib[f];
                    }
                }
            }
            if (A.obs_start) {
                const long long a0 = A.obs_start[s.ooff], a1 = A.obs_start[s.ooff + 1];
                for (long long q = a0 + tid; q < a1; q += WK_NT) {
                    const int idx = A.obs_idx[q], lj = A.obs_lj[q];
                    const int f = idx / g.ncell, li = idx - f * g.ncell - lj * g.ex;
                    const double rr = sm[st + f * FS + lj * P + li] - A.obs_y[q];
                    const double cq = A.obs_c[q];
                    ob += cq * rr * rr;
                    A.obs_r[q] = 2.0 * cq * rr;
                }
            }
        }
        wk_wait_read<0>();                      // level-0 stores have left shared memory
        bg = block_sum<WK_NT>(bg, red);
        sp = block_sum<WK_NT>(sp, red);
        pr = block_sum<WK_NT>(pr, red);
        ob = block_sum<WK_NT>(ob, red);         // (ends with a __syncthreads)

        // ---------------- per-lane column map of this tile
        int cj[K + 2];
#pragma unroll
        for (int j = 0; j < K + 2; ++j) { const int c = c0 - 1 + j; cj[j] = c < g.px ? c : g.px - 1; }
        bool tcol[K];
#pragma unroll
        for (int i = 0; i < K; ++i) tcol[i] = (c0 + i >= 3) && (c0 + i < 3 + g.ex);
        const bool injL = lane == 0, injR = (lane == 31) && (c0 + K == g.px - 2);
        const int gcp_src = (lane / 6) * 6 * WK_EWC + (lane % 6);
        const int gcp_dst = (lane / 6) * FS + ((lane % 6) < 3 ? (lane % 6) - 3 : g.ex + (lane % 6) - 3);
        const int nchunk = (g.ey + WK_EWC - 1) / WK_EWC;
        double obw = 0.0;                       // this lane's share of H (25b) over this warp's steps

        // ---------------- the steps of this warp
        for (int n = w; n < g.W; n += WK_NW) {
            const unsigned gs = gbase + (unsigned)n;
            const bool has_leader = n > 0;
            const unsigned need0 = (gs - 1u) << 10;
            const uint32_t a_lead = a_prog + 4u * lw;
            const double* gz = A.ghost + s.goff + (long long)n * 3 * g.nring;
            const double* ge = A.gedge + s.eoff + (long long)n * 2 * g.py;
            double* tout = A.traj + s.toff + (long long)(n + 1) * 3 * g.ncell;
            long long qcur = 0, qend = 0;
            if (A.obs_start) { qcur = A.obs_start[s.ooff + n + 1]; qend = A.obs_start[s.ooff + n + 2]; }
            const bool have_obs = qend > qcur;
            int p_lj = 0x7fffffff, p_idx = 0; double p_y = 0.0, p_c = 0.0;
            if (have_obs && qcur + lane < qend) {
                p_lj = A.obs_lj[qcur + lane]; p_idx = A.obs_idx[qcur + lane];
                p_y = A.obs_y[qcur + lane]; p_c = A.obs_c[qcur + lane];
            }
            auto issue_chunk = [&](int c) {     // lane 0: E/W ghost cells + edge u^a of tile rows [c*EWC, ...)
                const int r0 = c * WK_EWC;
                const int rows = g.ey - r0 < WK_EWC ? g.ey - r0 : WK_EWC;
                const int slot = c & 1;
                wk_mbar_expect(bar_ew + slot, (uint32_t)rows * (3u * 48u + 16u));
#pragma unroll
                for (int f = 0; f < 3; ++f)
                    wk_g2s(sm + I_EW + slot * 18 * WK_EWC + f * 6 * WK_EWC,
                           gz + (long long)f * g.nring + (g.gys + g.gyn) * g.px + r0 * 6, rows * 48u, bar_ew + slot);
                wk_g2s(sm + I_EDE + slot * 2 * WK_EWC, ge + (g.gys + g.gyn) * 2 + r0 * 2, rows * 16u, bar_ew + slot);
            };
            auto issue_ns = [&](bool north) {   // lane 0: the three ghost rows of one side + their edge u^a
                const int rows = north ? g.gyn : g.gys;
                const int roff = north ? g.gys : 0;
                wk_mbar_expect(bar_sn, (uint32_t)rows * (3u * g.px * 8u + 16u));
#pragma unroll
                for (int f = 0; f < 3; ++f)
                    wk_g2s(sm + I_SN + f * 3 * g.px, gz + (long long)f * g.nring + roff * g.px, rows * g.px * 8u, bar_sn);
                wk_g2s(sm + I_EDS + (north ? 8 : 0), ge + roff * 2, rows * 16u, bar_sn);
            };
            if (lane == 0) {
                if (g.gys) issue_ns(false); else if (g.gyn) issue_ns(true);
                issue_chunk(0);
                if (nchunk > 1) issue_chunk(1);
            }
            // row histories (names: 1 = row t-1, 2 = row t-2, ... at the start of tick t)
            double z1[3][K], z2[3][K], ha2[K], ua2[K], va2[K], va3[K], h13[K], h14[K], u13[K];
            double uaL2 = 0.0, uaR2 = 0.0;
#pragma unroll
            for (int i = 0; i < K; ++i) {
#pragma unroll
                for (int f = 0; f < 3; ++f) { z1[f][i] = 0.0; z2[f][i] = 0.0; }
                ha2[i] = ua2[i] = va2[i] = va3[i] = h13[i] = h14[i] = u13[i] = 0.0;
            }
            int prb = 0, prfs = 0;              // row reference of row t-1

            const int T = g.py + 3;
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                // ---- (0) row t becomes readable
                int rb = 0, rfs = 0;
                if (t < g.py) {
                    if (t < g.gys) {
                        if (t == 0) { wk_mbar_wait(bar_sn, par & 1u); par ^= 1u; }
                        rb = I_SN + t * g.px; rfs = 3 * g.px;
                    } else if (t < g.gys + g.ey) {
                        const int lj = t - g.gys;
                        const int slot = (lj / WK_EWC) & 1;
                        if ((lj % WK_EWC) == 0) { wk_mbar_wait(bar_ew + slot, (par >> (1 + slot)) & 1u); par ^= 2u << slot; }
                        if (has_leader) wk_wait_prog(a_lead, need0 + (unsigned)lj + 1u);
                        if (lane < 18)
                            sm[st + lj * P + gcp_dst] = sm[I_EW + slot * 18 * WK_EWC + (lj % WK_EWC) * 6 + gcp_src];
                        __syncwarp();
                        rb = st + lj * P - 3; rfs = FS;
                    } else {
                        if (t == g.gys + g.ey) { wk_mbar_wait(bar_sn, par & 1u); par ^= 1u; }
                        rb = I_SN + (t - g.gys - g.ey) * g.px; rfs = 3 * g.px;
                    }
                }
                // before this warp overwrites the last tile row: the leader's stores of it have left
                if (has_leader && t == g.gys + g.ey + 2) wk_wait_prog(a_lead, need0 + 1023u);

                // ---- (1) loads: own columns of row t, E/W halo of row t-1
                double z0[3][K], hz[3][2];
                if (t < g.py) {
#pragma unroll
                    for (int f = 0; f < 3; ++f)
#pragma unroll
                        for (int i = 0; i < K; ++i) z0[f][i] = sm[rb + f * rfs + cj[i + 1]];
                } else {
                    const double sg = (t == g.py && g.wn) ? -1.0 : 1.0;     // virtual mirrored row py
#pragma unroll
                    for (int i = 0; i < K; ++i) { z0[0][i] = z1[0][i]; z0[1][i] = z1[1][i]; z0[2][i] = sg * z1[2][i]; }
                }
                if (t >= 1 && t <= g.py) {
#pragma unroll
                    for (int f = 0; f < 3; ++f) { hz[f][0] = sm[prb + f * prfs + cj[0]]; hz[f][1] = sm[prb + f * prfs + cj[K + 1]]; }
                } else {
#pragma unroll
                    for (int f = 0; f < 3; ++f) { hz[f][0] = 0.0; hz[f][1] = 0.0; }
                }
                if (g.ws) {                      // virtual mirrored row -1 (R4)
                    if (t == 1) {
#pragma unroll
                        for (int i = 0; i < K; ++i) { z2[0][i] = z1[0][i]; z2[1][i] = z1[1][i]; z2[2][i] = -z1[2][i]; }
                    }
                    if (t == 2) {
#pragma unroll
                        for (int i = 0; i < K; ++i) va3[i] = -va2[i];
                    }
                    if (t == 3) {
#pragma unroll
                        for (int i = 0; i < K; ++i) h14[i] = h13[i];
                    }
                }

                // ---- (2) stage A on row t-1
                double ha1[K], ua1[K], va1[K], uaL1 = 0.0, uaR1 = 0.0;
                if (t >= 1 && t <= g.py) {
                    const double dtcz1 = tab[t * 8 + WK_T_DTCZ];
#pragma unroll
                    for (int i = 0; i < K; ++i) {
                        const double cu = dtcz1 * z1[1][i], cv = dtcm * z1[2][i];
                        double xa[3];
#pragma unroll
                        for (int f = 0; f < 3; ++f) {
                            const double xE = i < K - 1 ? z1[f][i + 1 < K ? i + 1 : i] : hz[f][1];
                            const double xW = i > 0 ? z1[f][i > 0 ? i - 1 : 0] : hz[f][0];
                            xa[f] = mm_stageA(z1[f][i], xE, xW, z0[f][i], z2[f][i], cu, cv, kap);
                        }
                        ha1[i] = xa[0]; ua1[i] = xa[1]; va1[i] = xa[2];
                    }
                    uaL1 = wk_up(ua1[K - 1]); uaR1 = wk_dn(ua1[0]);
                    // frozen u^a of the ghost columns 1 and px-2 of row t-1 (xk_edge_ua)
                    const int r1 = t - 1;
                    int ie;
                    if (r1 < g.gys) ie = I_EDS + r1 * 2;
                    else if (r1 < g.gys + g.ey) { const int l1 = r1 - g.gys; ie = I_EDE + ((l1 / WK_EWC) & 1) * 2 * WK_EWC + (l1 % WK_EWC) * 2; }
                    else ie = I_EDS + 8 + (r1 - g.gys - g.ey) * 2;
                    if (injL) uaL1 = sm[ie];
                    if (injR) uaR1 = sm[ie + 1];
                } else {
                    const double sg = (t == g.py + 1 && g.wn) ? -1.0 : 0.0;  // virtual row py: v^a mirrored
#pragma unroll
                    for (int i = 0; i < K; ++i) { ha1[i] = 0.0; ua1[i] = 0.0; va1[i] = sg * va2[i]; }
                }

                // ---- (3) h^1 and u^1 on row t-2
                double h12[K], u12[K];
                if (t >= 2 && t <= g.py + 1) {
                    const double* tb = tab + (t - 1) * 8;
                    const double dtcz2 = tb[WK_T_DTCZ], gdtcz2 = tb[WK_T_GDTCZ], dtf2 = tb[WK_T_DTF], dtt2 = tb[WK_T_DTT];
                    const double rp2 = tb[WK_T_RP], rm2 = tb[WK_T_RM];
#pragma unroll
                    for (int i = 0; i < K; ++i) {
                        const double uE = i < K - 1 ? ua2[i + 1 < K ? i + 1 : i] : uaR2;
                        const double uW = i > 0 ? ua2[i > 0 ? i - 1 : 0] : uaL2;
                        h12[i] = mm_h1(ha2[i], mm_div(uE, uW, va1[i], va3[i], dtcz2, dtcm, rp2, rm2));
                    }
                    const double hL = wk_up(h12[K - 1]), hR = wk_dn(h12[0]);
#pragma unroll
                    for (int i = 0; i < K; ++i) {
                        const double hE = i < K - 1 ? h12[i + 1 < K ? i + 1 : i] : hR;
                        const double hW = i > 0 ? h12[i > 0 ? i - 1 : 0] : hL;
                        u12[i] = mm_u1(ua2[i], va2[i], hE, hW, gdtcz2, dtf2, dtt2);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < K; ++i) { h12[i] = (t == g.py + 2 && g.wn) ? h13[i] : 0.0; u12[i] = 0.0; }
                }

                // ---- (4) v^1 on row t-3: row t-3 of Z^{n+1} is complete
                if (t >= 3) {
                    const int r3 = t - 3;
                    const double dtf3 = tab[(t - 2) * 8 + WK_T_DTF], dtt3 = tab[(t - 2) * 8 + WK_T_DTT];
                    if (r3 >= g.gys && r3 < g.gys + g.ey) {
                        const int lj = r3 - g.gys;
                        const int ob0 = st + lj * P + c0 - 3;
#pragma unroll
                        for (int i = 0; i < K; ++i) {
                            const double v1 = mm_v1(va3[i], u13[i], h12[i], h14[i], gdtcm, dtf3, dtt3);
                            if (tcol[i]) { sm[ob0 + i] = h13[i]; sm[ob0 + FS + i] = u13[i]; sm[ob0 + 2 * FS + i] = v1; }
                        }
                        wk_fence_async();
                        __syncwarp();
                        if (lane == 0) {
#pragma unroll
                            for (int f = 0; f < 3; ++f)
                                wk_s2g(tout + (long long)f * g.ncell + lj * g.ex, sm + st + f * FS + lj * P, g.ex * 8u);
                            wk_commit();
                        }
                        // H (25b) at level n+1 on this row: misfit, its cost, and the adjoint forcing r
                        if (have_obs) {
                            for (;;) {
                                const unsigned mm = __ballot_sync(0xffffffffu, p_lj == lj);
                                const int cnt = __popc(mm);
                                if (lane < cnt) {
                                    const int f = p_idx / g.ncell, li = p_idx - f * g.ncell - lj * g.ex;
                                    const double rr = sm[st + f * FS + lj * P + li] - p_y;
                                    obw += p_c * rr * rr;
                                    A.obs_r[qcur + lane] = 2.0 * p_c * rr;
                                }
                                if (cnt == 0) break;
                                qcur += cnt;
                                p_lj = 0x7fffffff;
                                if (qcur + lane < qend) {
                                    p_lj = A.obs_lj[qcur + lane]; p_idx = A.obs_idx[qcur + lane];
                                    p_y = A.obs_y[qcur + lane]; p_c = A.obs_c[qcur + lane];
                                }
                                if (cnt < 32) break;
                            }
                        }
                        if (lane == 0) {
                            wk_wait_read<1>();   // every store but the one just issued has left shared memory
                            wk_publish(a_prog + 4u * w, (gs << 10) + (unsigned)lj + 1u);
                        }
                    }
                }

                // ---- (5) refills: N ghost rows after the S rows are consumed; next E/W chunk
                if (t >= 1 && t <= g.py) {
                    const int r1 = t - 1;
                    if (g.gys && g.gyn && r1 == g.gys - 1) { __syncwarp(); if (lane == 0) issue_ns(true); }
                    if (r1 >= g.gys && r1 < g.gys + g.ey) {
                        const int l1 = r1 - g.gys;
                        if ((l1 % WK_EWC) == WK_EWC - 1 && l1 / WK_EWC + 2 < nchunk) { __syncwarp(); if (lane == 0) issue_chunk(l1 / WK_EWC + 2); }
                    }
                }

                // ---- (6) rotate the row histories
#pragma unroll
                for (int i = 0; i < K; ++i) {
#pragma unroll
                    for (int f = 0; f < 3; ++f) { z2[f][i] = z1[f][i]; z1[f][i] = z0[f][i]; }
                    ha2[i] = ha1[i]; ua2[i] = ua1[i]; va3[i] = va2[i]; va2[i] = va1[i];
                    h14[i] = h13[i]; h13[i] = h12[i]; u13[i] = u12[i];
                }
                uaL2 = uaL1; uaR2 = uaR1;
                prb = rb; prfs = rfs;
            }
            // step done: all its stores have left shared memory
            if (lane == 0) { wk_wait_read<0>(); wk_publish(a_prog + 4u * w, (gs << 10) + 1023u); }
            __syncwarp();
        }
        // ---------------- reduction of the cost terms (fixed order: lanes, then warps)
        for (int o = 16; o > 0; o >>= 1) obw += __shfl_down_sync(0xffffffffu, obw, o);
        if (lane == 0) wpart[w] = obw;
        __syncthreads();
        double su = 0.0;
        if (s.jw < A.geo.q - 1) {               // (25c) successor window: Z^W against its frozen control
            const double* xn = A.xfrozen + A.subs[k + A.geo.p1 * A.geo.p2].coff;
            for (int c = tid; c < g.ncell; c += WK_NT) {
                const int lj = c / g.ex, li = c - lj * g.ex;
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    const double dv = sm[st + f * FS + lj * P + li] - xn[(long long)f * g.ncell + c];
                    su += dv * dv * A.cp.ib[f];
                }
            }
        }
        su = block_sum<WK_NT>(su, red);
        if (tid == 0) {
            double obt = ob;
            for (int q = 0; q < WK_NW; ++q) obt += wpart[q];
            const double v[5] = { bg, obt, A.cp.mu * sp, A.cp.mu * pr, A.cp.mu * su };
            double tot = 0.0;
            for (int q = 0; q < 5; ++q) { A.parts[k * 5 + q] = v[q]; tot += v[q]; }
            A.J[k] = tot;
        }
        gbase += (unsigned)g.W + 1u;
    }
}
